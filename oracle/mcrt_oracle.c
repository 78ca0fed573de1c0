/*
 * mcrt_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-file CPU implementation (fp64, no blocking, no fusion) of the photon-packet
 * transport of Heymann & Siebenmorgen, "GPU-based Monte Carlo dust radiative transfer scheme applied
 * to AGN" (arxiv 1203.2941; text in /root/reference/PAPER.md).  It exists only so that tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs can check and time the
 * CUDA path against it.  It shares no code, header, table generator or constant with the CUDA
 * library under paper_1203_2941_b200/csrc/, and the product never calls it.
 *
 * The method is a stochastic simulation, so the oracle is the algorithm written out step by step in
 * the paper's order, with a fixed counter-based random-number contract so that a packet's trajectory
 * depends only on (seed, packet id, temperature-index field).  Each function cites the passage it
 * follows; where the paper is silent the reading is the one listed in DESIGN.md ("Readings").
 *
 * Parity pins (tests/test_oracle_pins.py): Philox known-answer vectors, DDA vs brute-force slab
 * intersections, exp(-tau) transmission, Henyey-Greenstein moments, isotropy, exact packet/energy
 * conservation, constant-albedo ratio, optically thin temperature, Planck/zeta closed forms,
 * 2x2x2 brute-force quadrature, per-cell redraw equivalence (paper fn. 1), epoch vs serial B&W (also at the
 * plateau-epoch shape of the default schedule, P12b), the explicit ln / sin / cos against libm and against
 * multi-precision values, the frozen-T sweep against the closed-form T(r) and the Eq. 5 mean photon energy
 * (P16), the SED flux conversion and E = k xi against L and the blackbody shape (P17), the position after
 * interactions against the random-flight second moment 2 l^2 / [(1-a)(1-a g)] (P18).
 * Parity UNPINNED: agreement with DUSTY / Kruegel / Pascucci benchmark SEDs,
 * whose data are not available here.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).  -ffp-contract=off
 * matters: every product/sum below is rounded separately, exactly as written.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018 / SI-2019 exact constants in cgs (reading Q15). */
static const double ORC_H = 6.62607015e-27;  /* erg s   */
static const double ORC_K = 1.380649e-16;    /* erg / K */
static const double ORC_C = 2.99792458e10;   /* cm / s  */
static const double ORC_FOUR_PI = 12.566370614359172953850573533118;

/* ------------------------------------------------------------------------------------------------
 * O2  Random numbers.  Philox-4x32-10 (Salmon, Moraes, Dror & Shaw 2011): 10 rounds, multipliers
 * 0xD2511F53 / 0xCD9E8D57, Weyl key increments 0x9E3779B9 / 0xBB67AE85.  Replaces the paper's
 * per-thread Mersenne Twister streams (Sect. 3.4) -- north_star item (1).
 * ---------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* One block -> two uniforms strictly inside (0,1) (reading Q3): u52 = top 52 bits of (w_a*2^32+w_b),
 * zeta = (2*u52 + 1) * 2^-53.  key = (seed lo, seed hi); counter = (pid lo, pid hi, draw index, pass). */
void orc_uniforms(uint64_t seed, uint64_t pid, uint32_t draw, uint32_t pass, double out[2])
{
    uint32_t ctr[4] = { (uint32_t)pid, (uint32_t)(pid >> 32), draw, pass };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    uint64_t a = (((uint64_t)w[0] << 32) | (uint64_t)w[1]) >> 12;
    uint64_t b = (((uint64_t)w[2] << 32) | (uint64_t)w[3]) >> 12;
    out[0] = (double)(2 * a + 1) * 0x1.0p-53;
    out[1] = (double)(2 * b + 1) * 0x1.0p-53;
}

/* ------------------------------------------------------------------------------------------------
 * O1  Tables.
 * ---------------------------------------------------------------------------------------------- */
/* Planck function B_nu(T), erg s^-1 cm^-2 Hz^-1 sr^-1 (Eq. 4). */
double orc_planck(double nu, double T)
{
    double x = ORC_H * nu / (ORC_K * T);
    return 2.0 * ORC_H * nu * nu * nu / (ORC_C * ORC_C) / expm1(x);
}

/* dB_nu/dT (Eq. 10): 2 h^2 nu^4 / (c^2 k T^2) * e^-x / (1 - e^-x)^2, x = h nu / k T. */
double orc_dplanck_dT(double nu, double T)
{
    double x = ORC_H * nu / (ORC_K * T);
    double em = exp(-x);
    double om = -expm1(-x);
    return 2.0 * ORC_H * ORC_H * nu * nu * nu * nu / (ORC_C * ORC_C * ORC_K * T * T) * em / (om * om);
}

/* Bin widths: bin j spans the geometric means of nu_j with its neighbours; the two end bins are
 * extrapolated with the neighbouring ratio (reading Q15; the paper only says a bin lies between
 * nu_j and nu_j+1). */
void orc_bin_widths(int nf, const double *nu, double *dnu)
{
    for (int j = 0; j < nf; ++j) {
        double lo = (j == 0) ? nu[0] * sqrt(nu[0] / nu[1]) : sqrt(nu[j - 1] * nu[j]);
        double hi = (j == nf - 1) ? nu[nf - 1] * sqrt(nu[nf - 1] / nu[nf - 2]) : sqrt(nu[j] * nu[j + 1]);
        dnu[j] = hi - lo;
    }
}

/* Running sum from the lowest frequency divided by the total; last entry forced to exactly 1.
 * Returns the total.  A row with zero total becomes (0,...,0,1). */
static double cumulative(int n, const double *w, double *cdf)
{
    double tot = 0.0;
    for (int j = 0; j < n; ++j) tot += w[j];
    double run = 0.0;
    for (int j = 0; j < n; ++j) {
        run += w[j];
        cdf[j] = (tot > 0.0) ? run / tot : 0.0;
    }
    cdf[n - 1] = 1.0;
    return tot;
}

/* Smallest index j with cdf[j] >= z ("the shortest frequency nu' for which the cumulative reaches
 * zeta", Eq. 5, 116-118 Eq. 10; reading Q17). */
int orc_lower_bound(const double *cdf, int n, double z)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        int mid = (lo + hi) / 2;
        if (cdf[mid] >= z) hi = mid; else lo = mid + 1;
    }
    return lo;
}

typedef struct {
    int nx, ny, nz, ns, nf, nT, ndir;
    double h;              /* cell size, cm */
    float *rho;            /* [nz][ny][nx] */
    uint8_t *sp;           /* [nz][ny][nx] */
    double *nu, *dnu;      /* [nf] */
    double *kabs, *ksca, *g; /* [ns][nf] */
    double *Tg;            /* [nT] */
    double *mu_edges;      /* [ndir+1] */
    double L;              /* erg/s */
    double pos[3];         /* source position in cell units */
    /* tables (O1) */
    double *kext_h;        /* (kabs+ksca)*h : optical depth per unit density per cell length */
    double *kabs_h;        /* kabs*h */
    double *albedo;        /* ksca/(ksca+kabs) */
    double *J;             /* [ns][nT]  sum_j kabs B_j(T) dnu_j, left side of Eq. 4 */
    double *cdfB;          /* [ns][nT][nf], Eq. 5 */
    double *cdfdB;         /* [ns][nT][nf], Eq. 10 */
    double *srccdf;        /* [nf] */
    /* NEXT-3 sub-cubes (orc_set_subgrid): refined cubes hold subR^3 sub-cubes each, numbered nc + block*subR^3 + local */
    int subR, n_sub;
    int32_t *sub_of_cell;  /* [nc] block number of a refined cube, -1 otherwise */
    float *sub_rho;        /* [n_sub][subR^3] (z, y, x) */
    uint8_t *sub_sp;
    /* NEXT-3 dust mixtures (orc_set_mixtures): with n_mix > 0 the species byte of a cell names a MIXTURE of one or
     * two of the ns materials, and kext_h / kabs_h / albedo above have n_mix rows (ntab = rows of those tables) */
    int ntab, n_mix;
    int32_t *mx_ncomp;     /* [n_mix] 1 or 2 components */
    int32_t *mx_mat;       /* [n_mix][2] material of each component */
    double *mx_frac;       /* [n_mix][2] mass fraction of each component */
    double *mx_S0, *mx_A0; /* [n_mix][nf] event thresholds (see orc_set_mixtures) */
    double *mx_kabs1_h;    /* [n_mix][nf] f_1 kabs_1 h of the second component (0 without one) */
} orc_ctx;

orc_ctx *orc_create(int nx, int ny, int nz, double h, const float *rho, const uint8_t *sp, int ns,
                    int nf, const double *nu, const double *kabs, const double *ksca, const double *g,
                    int nT, const double *Tg, double L, double Tstar, const double *Lnu_w,
                    const double pos_cm[3], int ndir, const double *mu_edges)
{
    orc_ctx *C = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    size_t nc = (size_t)nx * ny * nz;
    C->nx = nx; C->ny = ny; C->nz = nz; C->ns = ns; C->nf = nf; C->nT = nT; C->ndir = ndir; C->h = h; C->L = L;
    C->ntab = ns;
    C->rho = (float *)malloc(nc * sizeof(float));       memcpy(C->rho, rho, nc * sizeof(float));
    C->sp = (uint8_t *)malloc(nc);                      memcpy(C->sp, sp, nc);
    C->nu = (double *)malloc(nf * sizeof(double));      memcpy(C->nu, nu, nf * sizeof(double));
    C->dnu = (double *)malloc(nf * sizeof(double));
    size_t nsf = (size_t)ns * nf;
    C->kabs = (double *)malloc(nsf * sizeof(double));   memcpy(C->kabs, kabs, nsf * sizeof(double));
    C->ksca = (double *)malloc(nsf * sizeof(double));   memcpy(C->ksca, ksca, nsf * sizeof(double));
    C->g = (double *)malloc(nsf * sizeof(double));      memcpy(C->g, g, nsf * sizeof(double));
    C->Tg = (double *)malloc(nT * sizeof(double));      memcpy(C->Tg, Tg, nT * sizeof(double));
    C->mu_edges = (double *)malloc((ndir + 1) * sizeof(double));
    memcpy(C->mu_edges, mu_edges, (ndir + 1) * sizeof(double));
    for (int a = 0; a < 3; ++a) C->pos[a] = pos_cm[a] / h;

    orc_bin_widths(nf, nu, C->dnu);
    C->kext_h = (double *)malloc(nsf * sizeof(double));
    C->kabs_h = (double *)malloc(nsf * sizeof(double));
    C->albedo = (double *)malloc(nsf * sizeof(double));
    for (size_t i = 0; i < nsf; ++i) {
        double kext = kabs[i] + ksca[i];
        C->kext_h[i] = kext * h;
        C->kabs_h[i] = kabs[i] * h;
        C->albedo[i] = (kext > 0.0) ? ksca[i] / kext : 0.0;
    }
    C->J = (double *)malloc((size_t)ns * nT * sizeof(double));
    C->cdfB = (double *)malloc((size_t)ns * nT * nf * sizeof(double));
    C->cdfdB = (double *)malloc((size_t)ns * nT * nf * sizeof(double));
    double *w = (double *)malloc(nf * sizeof(double));
    for (int s = 0; s < ns; ++s)
        for (int m = 0; m < nT; ++m) {
            size_t row = ((size_t)s * nT + m) * nf;
            for (int j = 0; j < nf; ++j) w[j] = kabs[s * nf + j] * orc_planck(nu[j], Tg[m]) * C->dnu[j];
            C->J[(size_t)s * nT + m] = cumulative(nf, w, C->cdfB + row);
            for (int j = 0; j < nf; ++j) w[j] = kabs[s * nf + j] * orc_dplanck_dT(nu[j], Tg[m]) * C->dnu[j];
            cumulative(nf, w, C->cdfdB + row);
        }
    /* source: equal-energy packets drawn through the cumulative source spectrum (PAPER.md:39-45,
     * Eq. 1; reading Q1/Q2: one draw through the CDF on the shared grid). */
    C->srccdf = (double *)malloc(nf * sizeof(double));
    for (int j = 0; j < nf; ++j)
        w[j] = ((Tstar > 0.0) ? orc_planck(nu[j], Tstar) : Lnu_w[j]) * C->dnu[j];
    cumulative(nf, w, C->srccdf);
    free(w);
    return C;
}

void orc_destroy(orc_ctx *C)
{
    if (!C) return;
    free(C->rho); free(C->sp); free(C->nu); free(C->dnu); free(C->kabs); free(C->ksca); free(C->g);
    free(C->Tg); free(C->mu_edges); free(C->kext_h); free(C->kabs_h); free(C->albedo); free(C->J);
    free(C->cdfB); free(C->cdfdB); free(C->srccdf);
    free(C->sub_of_cell); free(C->sub_rho); free(C->sub_sp);
    free(C->mx_ncomp); free(C->mx_mat); free(C->mx_frac); free(C->mx_S0); free(C->mx_A0); free(C->mx_kabs1_h);
    free(C);
}

/* NEXT-3: per-cell dust mixtures with per-material temperatures.  PAPER.md:17 "equilibrium
 * temperatures of two populations of large grains", "different grain materials", "the total
 * number of absorbed photon packets per particle and cell is used to calculate the temperature of each material".
 * The paper gives no formulas for the mixture; readings Q34-Q36:
 *   Q34  a cell of mixture x holds its components c = 0, 1 (materials m_c) with mass fractions f_c of the cell's
 *        density; extinction adds up:  kext_x = (f_0 kabs_0 + f_0 ksca_0) + (f_1 kabs_1 + f_1 ksca_1)   (Eq. 2)
 *   Q35  the ONE uniform number that decides scattering against absorption also decides which
 *        component interacts, each in proportion to its share of kext_x:
 *          z < S0           scattered by component 0   (its g in the HG function)   S0 = f_0 ksca_0 / kext_x
 *          z < albedo       scattered by component 1                                albedo = (f_0 ksca_0 + f_1 ksca_1) / kext_x
 *          z < A0           absorbed by component 0                                 A0 = ((f_0 ksca_0 + f_1 ksca_1) + f_0 kabs_0) / kext_x
 *          else             absorbed by component 1
 *   Q36  every component has its own absorption count, Lucy tally (f_c kabs_c rho ds per traversal) and
 *        temperature: Eq. 4 with the component's material and its mass rho_i f_c V_i; an absorbed packet is
 *        re-emitted from the absorbing component's Eq. 10 / Eq. 5 row at that component's temperature.
 * Returns 0, -1 on bad arguments.  Call before orc_state_create. */
int orc_set_mixtures(orc_ctx *C, int n_mix, const int32_t *ncomp, const int32_t *mat, const double *frac)
{
    if (n_mix < 1 || n_mix > 255) return -1;
    for (int x = 0; x < n_mix; ++x) {
        if (ncomp[x] < 1 || ncomp[x] > 2) return -1;
        double tot = 0.0;
        for (int c = 0; c < ncomp[x]; ++c) {
            if (mat[2 * x + c] < 0 || mat[2 * x + c] >= C->ns || !(frac[2 * x + c] > 0.0)) return -1;
            tot += frac[2 * x + c];
        }
        if (fabs(tot - 1.0) > 1e-12) return -1;
    }
    const int nf = C->nf;
    const size_t n = (size_t)n_mix * nf;
    C->n_mix = n_mix; C->ntab = n_mix;
    C->mx_ncomp = (int32_t *)malloc(n_mix * sizeof(int32_t));
    C->mx_mat = (int32_t *)calloc(2 * (size_t)n_mix, sizeof(int32_t));
    C->mx_frac = (double *)calloc(2 * (size_t)n_mix, sizeof(double));
    C->mx_S0 = (double *)calloc(n, sizeof(double));
    C->mx_A0 = (double *)calloc(n, sizeof(double));
    C->mx_kabs1_h = (double *)calloc(n, sizeof(double));
    free(C->kext_h); free(C->kabs_h); free(C->albedo);
    C->kext_h = (double *)malloc(n * sizeof(double));
    C->kabs_h = (double *)malloc(n * sizeof(double));
    C->albedo = (double *)malloc(n * sizeof(double));
    for (int x = 0; x < n_mix; ++x) {
        C->mx_ncomp[x] = ncomp[x];
        for (int c = 0; c < ncomp[x]; ++c) { C->mx_mat[2 * x + c] = mat[2 * x + c]; C->mx_frac[2 * x + c] = frac[2 * x + c]; }
        for (int j = 0; j < nf; ++j) {
            const size_t i = (size_t)x * nf + j;
            const int m0 = mat[2 * x];
            if (ncomp[x] == 1) {      /* the material itself: the same arithmetic as without mixtures */
                double kext = C->kabs[m0 * nf + j] + C->ksca[m0 * nf + j];
                C->kext_h[i] = kext * C->h;
                C->kabs_h[i] = C->kabs[m0 * nf + j] * C->h;
                C->albedo[i] = (kext > 0.0) ? C->ksca[m0 * nf + j] / kext : 0.0;
                C->mx_S0[i] = C->albedo[i]; C->mx_A0[i] = 1.0;
            } else {
                const int m1 = mat[2 * x + 1];
                double ka0 = frac[2 * x] * C->kabs[m0 * nf + j], ks0 = frac[2 * x] * C->ksca[m0 * nf + j];
                double ka1 = frac[2 * x + 1] * C->kabs[m1 * nf + j], ks1 = frac[2 * x + 1] * C->ksca[m1 * nf + j];
                double kext = (ka0 + ks0) + (ka1 + ks1);
                C->kext_h[i] = kext * C->h;
                C->kabs_h[i] = ka0 * C->h;
                C->mx_kabs1_h[i] = ka1 * C->h;
                C->mx_S0[i] = (kext > 0.0) ? ks0 / kext : 0.0;
                C->albedo[i] = (kext > 0.0) ? (ks0 + ks1) / kext : 0.0;
                C->mx_A0[i] = (kext > 0.0) ? ((ks0 + ks1) + ka0) / kext : 1.0;
            }
        }
    }
    return 0;
}

/* NEXT-3, one level of refinement: "Each cube is divided into an arbitrary number of sub-cubes of volume
 * V_i and constant density rho_i ... The subdivision of cubes allows a finer sampling whenever required".
 * Reading Q40: a refined cube holds R x R x R equal sub-cubes, R = 2, 4 or 8 the same for all refined cubes
 * of a grid, each with its own density and species; a packet crosses them with the same cell walk on the lattice of
 * sub-cube faces (face coordinates c + k/R are exact doubles), every sub-cube is a cell of its own for optical depth,
 * tallies, absorption counts and temperature (Eq. 4 with V = (h/R)^3).  Cell numbers of sub-cubes: nc + block R^3 +
 * (gz R + gy) R + gx.  With every cube refined the run IS the run on the (n R)^3 uniform grid, bit for bit (pin P24).
 * cube[n_sub]: cell index of every refined cube; rho_sub / sp_sub [n_sub][R^3].  Call before orc_state_create. */
int orc_set_subgrid(orc_ctx *C, int R, int n_sub, const int64_t *cube, const float *rho_sub, const uint8_t *sp_sub)
{
    if ((R != 2 && R != 4 && R != 8) || n_sub < 1 || C->n_mix) return -1;
    size_t nc = (size_t)C->nx * C->ny * C->nz, R3 = (size_t)R * R * R;
    C->sub_of_cell = (int32_t *)malloc(nc * sizeof(int32_t));
    for (size_t i = 0; i < nc; ++i) C->sub_of_cell[i] = -1;
    for (int b = 0; b < n_sub; ++b) {
        if (cube[b] < 0 || (size_t)cube[b] >= nc || C->sub_of_cell[cube[b]] >= 0) return -1;
        C->sub_of_cell[cube[b]] = b;
    }
    for (size_t i = 0; i < n_sub * R3; ++i)
        if (!(rho_sub[i] >= 0.0f) || sp_sub[i] >= C->ns) return -1;
    C->sub_rho = (float *)malloc(n_sub * R3 * sizeof(float));  memcpy(C->sub_rho, rho_sub, n_sub * R3 * sizeof(float));
    C->sub_sp = (uint8_t *)malloc(n_sub * R3);                 memcpy(C->sub_sp, sp_sub, n_sub * R3);
    C->subR = R; C->n_sub = n_sub;
    return 0;
}
/* all cells, sub-cubes included: count, density (0 for a refined cube itself: its dust is in its sub-cubes), species */
static inline size_t cells_total(const orc_ctx *C)
{
    size_t nc = (size_t)C->nx * C->ny * C->nz;
    return C->subR ? nc + (size_t)C->n_sub * C->subR * C->subR * C->subR : nc;
}
static inline double cell_rho(const orc_ctx *C, size_t ci)
{
    size_t nc = (size_t)C->nx * C->ny * C->nz;
    if (ci >= nc) return (double)C->sub_rho[ci - nc];
    if (C->subR && C->sub_of_cell[ci] >= 0) return 0.0;
    return (double)C->rho[ci];
}
static inline int cell_sp(const orc_ctx *C, size_t ci)
{
    size_t nc = (size_t)C->nx * C->ny * C->nz;
    return ci >= nc ? C->sub_sp[ci - nc] : C->sp[ci];
}
/* Eq. 4's xi / (4 pi V) for cell ci: V = h^3, or (h/R)^3 for a sub-cube (computed like the uniform grid of that cell size) */
static inline double cell_fac(const orc_ctx *C, size_t ci, double xi)
{
    size_t nc = (size_t)C->nx * C->ny * C->nz;
    double hh = ci >= nc ? C->h / (double)C->subR : C->h;
    return xi / (ORC_FOUR_PI * hh * hh * hh);
}

/* material and mass fraction of component c of the cell species x (without mixtures: the material x itself) */
static inline int comp_mat(const orc_ctx *C, int x, int c) { return C->n_mix ? C->mx_mat[2 * x + c] : x; }
static inline int comp_count(const orc_ctx *C, int x) { return C->n_mix ? C->mx_ncomp[x] : 1; }

/* table accessors for the pins */
void orc_get_tables(const orc_ctx *C, double *dnu, double *J, double *cdfB, double *cdfdB, double *albedo,
                    double *srccdf)
{
    if (dnu) memcpy(dnu, C->dnu, C->nf * sizeof(double));
    if (J) memcpy(J, C->J, (size_t)C->ns * C->nT * sizeof(double));
    if (cdfB) memcpy(cdfB, C->cdfB, (size_t)C->ns * C->nT * C->nf * sizeof(double));
    if (cdfdB) memcpy(cdfdB, C->cdfdB, (size_t)C->ns * C->nT * C->nf * sizeof(double));
    if (albedo) memcpy(albedo, C->albedo, (size_t)C->ns * C->nf * sizeof(double));
    if (srccdf) memcpy(srccdf, C->srccdf, C->nf * sizeof(double));
}

/* ------------------------------------------------------------------------------------------------
 * Elementary functions of the trajectory (reading Q28).
 * tau = -ln zeta and the azimuth phi = 2 pi zeta need ln, sin and cos.
 * Math libraries differ in the last ulp of these, and a clumpy medium amplifies an ulp into a different
 * trajectory, so the method's ln / sin / cos are DEFINED by the explicit fp64
 * algorithms below: only + - * / on doubles, every operation rounded separately, fixed order.  They are
 * accurate to 2 ulp (pinned against libm in tests/test_oracle_pins.py), which is physically irrelevant.
 * ---------------------------------------------------------------------------------------------- */
/* ln z for a positive normal double: z = m 2^e with m in (sqrt(1/2), sqrt(2)];
 * ln m = 2 atanh(s), s = (m-1)/(m+1), by its Taylor series up to s^25; ln 2 split in two parts. */
double orc_det_log(double z)
{
    uint64_t b;
    memcpy(&b, &z, 8);
    int e = (int)((b >> 52) & 0x7ffu) - 1023;
    b = (b & 0x000fffffffffffffull) | 0x3ff0000000000000ull;
    double m;
    memcpy(&m, &b, 8);
    if (m > 0x1.6a09e667f3bcdp+0) { m = m * 0.5; e += 1; }
    double f = m - 1.0;
    double s = f / (2.0 + f);
    double z2 = s * s;
    double p = 1.0 / 25.0;
    p = p * z2 + 1.0 / 23.0;
    p = p * z2 + 1.0 / 21.0;
    p = p * z2 + 1.0 / 19.0;
    p = p * z2 + 1.0 / 17.0;
    p = p * z2 + 1.0 / 15.0;
    p = p * z2 + 1.0 / 13.0;
    p = p * z2 + 1.0 / 11.0;
    p = p * z2 + 1.0 / 9.0;
    p = p * z2 + 1.0 / 7.0;
    p = p * z2 + 1.0 / 5.0;
    p = p * z2 + 1.0 / 3.0;
    double t = s * (z2 * p);
    double lm = 2.0 * s + 2.0 * t;
    double ed = (double)e;
    return (ed * 0x1.62e42fee00000p-1 + lm) + ed * 0x1.a39ef35793c76p-33;
}

/* sin and cos of 2 pi z, z in [0, 1): quarter turns q = round(4 z), remainder r = 4 z - q in [-1/2, 1/2]
 * (both exact), x = r pi/2, Taylor series of sin and cos up to x^19 and x^18, then the quadrant. */
void orc_det_sincos(double z, double *sn, double *cs)
{
    double a = 4.0 * z;
    double qd = floor(a + 0.5);
    double r = a - qd;
    double x = r * 0x1.921fb54442d18p+0;
    double x2 = x * x;
    double p = -1.0 / 121645100408832000.0;       /* -1/19! */
    p = p * x2 + 1.0 / 355687428096000.0;          /* +1/17! */
    p = p * x2 - 1.0 / 1307674368000.0;            /* -1/15! */
    p = p * x2 + 1.0 / 6227020800.0;               /* +1/13! */
    p = p * x2 - 1.0 / 39916800.0;                 /* -1/11! */
    p = p * x2 + 1.0 / 362880.0;                   /* +1/9!  */
    p = p * x2 - 1.0 / 5040.0;                     /* -1/7!  */
    p = p * x2 + 1.0 / 120.0;                      /* +1/5!  */
    p = p * x2 - 1.0 / 6.0;                        /* -1/3!  */
    double s = x + x * (x2 * p);
    double c = -1.0 / 6402373705728000.0;          /* -1/18! */
    c = c * x2 + 1.0 / 20922789888000.0;           /* +1/16! */
    c = c * x2 - 1.0 / 87178291200.0;              /* -1/14! */
    c = c * x2 + 1.0 / 479001600.0;                /* +1/12! */
    c = c * x2 - 1.0 / 3628800.0;                  /* -1/10! */
    c = c * x2 + 1.0 / 40320.0;                    /* +1/8!  */
    c = c * x2 - 1.0 / 720.0;                      /* -1/6!  */
    c = c * x2 + 1.0 / 24.0;                       /* +1/4!  */
    c = c * x2 - 0.5;                              /* -1/2!  */
    double co = 1.0 + x2 * c;
    int q = (int)qd & 3;
    if (q == 0) { *sn = s; *cs = co; }
    else if (q == 1) { *sn = co; *cs = -s; }
    else if (q == 2) { *sn = -s; *cs = -co; }
    else { *sn = -co; *cs = s; }
}

/* ------------------------------------------------------------------------------------------------
 * Directions.
 * ---------------------------------------------------------------------------------------------- */
/* phi = 2 pi zeta_1, cos(theta) = 1 - 2 zeta_2.  (Here zeta0 -> cos theta, zeta1 -> phi.) */
void orc_isotropic(double z0, double z1, double u[3])
{
    double mu = 1.0 - 2.0 * z0;
    double sp, cp;
    orc_det_sincos(z1, &sp, &cp);   /* phi = 2 pi z1 */
    double st = sqrt(1.0 - mu * mu);
    u[0] = st * cp;
    u[1] = st * sp;
    u[2] = mu;
}

/* O7 Henyey-Greenstein scattering (phase function Eq. 15).  The paper
 * gives only P_HG; the sampling is its analytic inversion (reading Q12), isotropic below |g| = 1e-6,
 * and the new direction is (theta, phi) about the old one (reading Q13). */
void orc_hg_scatter(double gg, double z0, double z1, const double u[3], double un[3])
{
    double mu;
    if (fabs(gg) <= 1e-6) {
        mu = 1.0 - 2.0 * z0;
    } else {
        double q = (1.0 - gg * gg) / (1.0 - gg + 2.0 * gg * z0);
        mu = (1.0 + gg * gg - q * q) / (2.0 * gg);
        if (mu > 1.0) mu = 1.0;
        if (mu < -1.0) mu = -1.0;
    }
    double sp, cp;
    orc_det_sincos(z1, &sp, &cp);   /* phi = 2 pi z1 */
    double st = sqrt(1.0 - mu * mu);
    double a0, a1, a2;
    if (fabs(u[2]) > 0.99999) {
        a0 = st * cp;
        a1 = st * sp;
        a2 = (u[2] > 0.0) ? mu : -mu;
    } else {
        double w = sqrt(1.0 - u[2] * u[2]);
        double iw = 1.0 / w;
        double t0 = u[0] * u[2] * cp - u[1] * sp;
        double t1 = u[1] * u[2] * cp + u[0] * sp;
        a0 = st * t0 * iw + u[0] * mu;
        a1 = st * t1 * iw + u[1] * mu;
        a2 = u[2] * mu - st * cp * w;
    }
    double inorm = 1.0 / sqrt(a0 * a0 + a1 * a1 + a2 * a2);
    un[0] = a0 * inorm;
    un[1] = a1 * inorm;
    un[2] = a2 * inorm;
}

/* ------------------------------------------------------------------------------------------------
 * O4  Cell walk.  The paper says only that a packet "enters a neighboring cell according to its
 * direction of travel"; the walk is the Amanatides-Woo voxel traversal (reading Q8):
 * per axis the parameter t of the next face, measured from the flight origin in cell units;
 * the axis with the smallest one is crossed next (ties x before y before z).  The parameter of a
 * face is always computed from the face coordinate itself, t = (f - p_a) * (1/u_a) (reading Q8,
 * DESIGN.md section 2): it is a function of the face alone, so the walk is the three-way merge of the
 * per-axis face sequences ordered by (t, axis) and carries no accumulated rounding.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    double tmax[3], inv[3], p[3];
    int step[3];
} orc_dda;

/* parameter of the face the packet leaves cell c_a through, along axis a */
static inline double dda_face_t(const orc_dda *D, int a, int c_a)
{
    if (D->step[a] == 0) return INFINITY;
    return ((double)(c_a + (D->step[a] > 0 ? 1 : 0)) - D->p[a]) * D->inv[a];
}

static void dda_setup(orc_dda *D, const double p[3], const double u[3], const int c[3])
{
    for (int a = 0; a < 3; ++a) {
        D->p[a] = p[a];
        D->step[a] = (u[a] > 0.0) ? 1 : ((u[a] < 0.0) ? -1 : 0);
        D->inv[a] = (D->step[a] != 0) ? 1.0 / u[a] : INFINITY;
        D->tmax[a] = dda_face_t(D, a, c[a]);
    }
}

/* cross the face of axis a: next cell, and the parameter of the face it will be left through */
static inline void dda_advance(orc_dda *D, int a, int c[3])
{
    c[a] += D->step[a];
    D->tmax[a] = dda_face_t(D, a, c[a]);
}

static inline int dda_axis(const orc_dda *D)
{
    if (D->tmax[0] <= D->tmax[1] && D->tmax[0] <= D->tmax[2]) return 0;
    if (D->tmax[1] <= D->tmax[2]) return 1;
    return 2;
}

/* start cell of a point (O3; reading Q9): floor(p) unless p sits on a face, then by direction sign */
static void start_cell(const double p[3], const double u[3], int c[3])
{
    for (int a = 0; a < 3; ++a) {
        double fl = floor(p[a]);
        if (p[a] != fl) c[a] = (int)fl;
        else c[a] = (u[a] >= 0.0) ? (int)fl : (int)fl - 1;
    }
}

/* Pin helper: list (cell, segment length) of a ray from p along u until it leaves the grid. */
int orc_dda_trace(int nx, int ny, int nz, const double p[3], const double u[3], int max_n,
                  int64_t *cells, double *ds_out)
{
    int c[3];
    int n[3] = { nx, ny, nz };
    start_cell(p, u, c);
    orc_dda D;
    dda_setup(&D, p, u, c);
    double t = 0.0;
    int cnt = 0;
    for (;;) {
        if (c[0] < 0 || c[0] >= n[0] || c[1] < 0 || c[1] >= n[1] || c[2] < 0 || c[2] >= n[2]) break;
        int a = dda_axis(&D);
        double tn = D.tmax[a];
        if (cnt < max_n) {
            cells[cnt] = ((int64_t)c[2] * ny + c[1]) * nx + c[0];
            ds_out[cnt] = tn - t;
        }
        ++cnt;
        t = tn;
        dda_advance(&D, a, c);
    }
    return cnt;
}

/* ------------------------------------------------------------------------------------------------
 * Run state and the packet routine.
 * ---------------------------------------------------------------------------------------------- */
enum { ORC_MODE_BW_EPOCH = 0, ORC_MODE_FROZEN_SWEEP = 1 };
enum { ORC_EV_EMIT = 0, ORC_EV_SCATTER = 1, ORC_EV_ABSORB = 2, ORC_EV_ESCAPE = 3 };

typedef struct {
    uint64_t hash;
    uint32_t crossings, scatterings, absorptions, escape_bin;
} orc_digest;

typedef struct {
    uint64_t packets, crossings, dusty_crossings, flights, scatterings, absorptions, escapes,
        direct_escapes, epochs, lucy_adds;
    int32_t fx_bits, overflow;
} orc_stats;

typedef struct {
    int32_t mode;            /* ORC_MODE_* */
    uint64_t B0, Bmax;       /* epoch schedule; 0 = defaults of O11 */
    int32_t n_sweeps;        /* frozen-T sweeps (mode 1) */
    int32_t sweep_T_from_lucy; /* 1: sweeps take T from the Lucy tally, 0: from counts */
    int32_t n_threads;       /* 1 = serial */
    int32_t absorb_and_stop; /* pin P10: an absorbed packet ends */
    int32_t per_cell_redraw; /* pin P11: new zeta on every cell entry, the paper's literal form */
    int32_t keep_fp64_lucy;  /* pin P14: also keep a compensated fp64 Lucy sum (serial only) */
    int32_t reset;           /* zero tallies first */
    uint32_t pass0;          /* RNG pass word of the B&W run */
    uint64_t pid0;           /* id of the first packet of this run (continuing a run with further packets) */
    uint64_t n_total;        /* the luminosity is split into this many packets, xi = L / n_total; 0 = n_packets */
    double growth;           /* epoch e+1 has min(floor(B_e * growth), Bmax) packets; 0 = 2 (O11) */
    uint32_t carry_K;        /* > 0: a packet is carried over to the next epoch after this many interactions in one epoch */
    uint32_t source_strata;  /* > 0: the source frequency is drawn stratified (Eq. 1): stratum = packet id mod source_strata */
    int32_t lucy_hybrid;     /* 1: the thresholded estimator of Sect. 3.1 / Eq. 9 (see orc_thin_cell, lucy_add) */
} orc_opts;

/* Sect. 3.1: "It is applied whenever the maximal optical depth of a cell i is smaller than 10^-2."
 * Reading Q37: the maximal optical depth of a cell is that of its longest chord, the diagonal, at the frequency of
 * its largest extinction: tau_max = sqrt(3) h rho_i max_nu (kabs + ksca). */
#define ORC_THIN_TAU 1e-2
static inline int orc_thin_cell(double rho_c, double kmax_diag) { return rho_c > 0.0 && rho_c * kmax_diag < ORC_THIN_TAU; }
/* Eq. 9: E_abs = (1 - e^-tau) xi for one traversal, tau the absorption optical depth of the chord (reading Q38: the
 * energy ABSORBED, so kabs only).  tau < 10^-2 here, and 1 - e^-tau is DEFINED as its series up to tau^5 in this
 * fixed order (truncation < 2 10^-13 relative), so that every implementation gets the same bits. */
static inline double orc_eq9(double tau)
{
    return tau * (1.0 - tau * (0.5 - tau * (1.0 / 6.0 - tau * (1.0 / 24.0 - tau * (1.0 / 120.0)))));
}

/* One stored scattering event ("The index of the cell, the frequency of the scattered photon and the
 * incoming direction is stored"): cell in [nz][ny][nx] order, slot of the frequency bin among the recorded ones,
 * incoming direction quantised to 16 bits per component, q_a = rint(32767 u_a). */
typedef struct orc_sca_event_s {
    uint32_t cell;
    uint16_t slot;
    int16_t q[3];
} orc_sca_event;

/* A packet carried over an epoch boundary: everything its continuation depends on.  The paper pauses packets with
 * more than 100 interactions in one cell once 80 % of the threads have finished, stores position and frequency and
 * resumes them at the end; which packets that hits depends on scheduling.  The deterministic
 * restatement (reading Q23): a packet that has had carry_K interactions within ONE epoch stops after the
 * carry_K-th (its new direction and frequency already drawn) and continues in the next epoch, from the same state
 * and with its own random stream, at that epoch's temperatures.  After the last epoch the carried packets run in
 * further epochs, with the budget doubled each time, until none is left. */
typedef struct {
    uint64_t pid, hash;
    double p[3], u[3];
    int32_t c[3], j;
    uint32_t d, ncross, nsca, nabs;
} orc_carry;

typedef struct {
    const orc_ctx *C;
    uint64_t *k, *kprev;     /* absorption counts */
    int64_t *Lfx;            /* Lucy path-length tally, fixed point (O9) */
    double *Lsum, *Lcmp;     /* compensated fp64 copy */
    uint16_t *tidx;          /* temperature index per cell (O11) */
    uint64_t *k1;            /* the same three for the second component of a mixture (NEXT-3), or NULL */
    int64_t *Lfx1;
    uint16_t *tidx1;
    double *kabs1_fx;
    const double *kmax_diag; /* lucy_hybrid: [ns] sqrt(3) h max_nu (kabs + ksca) per species, else NULL */
    uint64_t *sed, *sed_direct; /* [ndir][nf] */
    orc_digest *dig;         /* [n_packets] or NULL */
    double *kabs_fx;         /* kabs_h * 2^FX */
    const double *cdf;       /* cdfdB (B&W) or cdfB (sweeps) */
    uint64_t seed;
    uint32_t pass;
    int fx;
    uint64_t pid0_digest;
    uint32_t carry_K;        /* interaction budget of the current epoch (0 = none) */
    const orc_opts *o;
    /* scattering-event store: slot of each frequency bin (-1 = not recorded), list, fill count */
    const int32_t *sca_slot;
    struct orc_sca_event_s *sca_ev;
    uint64_t sca_cap, *sca_n;
} orc_run_t;

static inline void hash_mix(uint64_t *h, uint64_t w)
{
    *h = (*h ^ w) * 0x100000001B3ull;
}

static inline uint64_t event_word(int type, int j, uint64_t cell)
{
    return (uint64_t)type | ((uint64_t)j << 8) | (cell << 24);
}

/* O9 Lucy path-length tally: every traversed dusty cell receives kappa_abs*rho*h*ds (in units of the
 * packet energy), the linear form of PAPER.md:105 Eq. 9 (reading Q21), kept as a 64-bit fixed-point
 * integer so that the sum does not depend on the order of additions (integer atomics). */
static inline void lucy_add(orc_run_t *R, size_t ci, int sj, double rho_c, double ds, orc_stats *st)
{
    if (R->kmax_diag) {
        /* Sect. 3.1 as printed: only cells below the threshold are tallied, with Eq. 9 per traversal (readings Q37, Q38) */
        if (!orc_thin_cell(rho_c, R->kmax_diag[sj / R->C->nf])) return;
        double tau = R->kabs_fx[sj] * rho_c * ds * ldexp(1.0, -R->fx);
        int64_t q = (int64_t)llrint(ldexp(orc_eq9(tau), R->fx));
        __atomic_fetch_add(&R->Lfx[ci], q, __ATOMIC_RELAXED);
        st->lucy_adds++;
        return;
    }
    if (rho_c > 0.0) {
        double x = R->kabs_fx[sj] * rho_c * ds;
        int64_t q = (int64_t)llrint(x);
        __atomic_fetch_add(&R->Lfx[ci], q, __ATOMIC_RELAXED);
        st->lucy_adds++;
        if (R->Lfx1 && R->C->mx_ncomp[sj / R->C->nf] == 2) {   /* second component of a mixture (reading Q36) */
            int64_t q1 = (int64_t)llrint(R->kabs1_fx[sj] * rho_c * ds);
            __atomic_fetch_add(&R->Lfx1[ci], q1, __ATOMIC_RELAXED);
        }
        if (R->Lsum) { /* Kahan */
            double y = R->C->kabs_h[sj] * rho_c * ds - R->Lcmp[ci];
            double tt = R->Lsum[ci] + y;
            R->Lcmp[ci] = (tt - R->Lsum[ci]) - y;
            R->Lsum[ci] = tt;
        }
    }
}

/* Follows one packet (a new one, or one carried over: `resume`) until it escapes -- returns 0 -- or until its
 * interaction budget of this epoch is used up: its state is written to *park and 1 is returned. */
static int run_packet(orc_run_t *R, uint64_t pid, orc_stats *st, const orc_carry *resume, orc_carry *park)
{
    const orc_ctx *C = R->C;
    const int nf = C->nf;
    const int n[3] = { C->nx, C->ny, C->nz };
    uint32_t d = 0;
    double z[2];
    double p[3], u[3];
    int c[3];
    uint32_t ncross = 0, nsca = 0, nabs = 0, nint = 0;
    uint64_t hash = 0xCBF29CE484222325ull;
    int j;
    /* sub-cubes (orc_set_subgrid): the sub-cube g of cube c the packet is in, if g_ok */
    const int subR = C->subR;
    const size_t nc0 = (size_t)n[0] * n[1] * n[2], R3 = (size_t)subR * subR * subR;
    int g[3] = { 0, 0, 0 }, g_ok = 0;

    if (resume) {
        pid = resume->pid; hash = resume->hash; j = resume->j; d = resume->d;
        ncross = resume->ncross; nsca = resume->nsca; nabs = resume->nabs;
        for (int a = 0; a < 3; ++a) { p[a] = resume->p[a]; u[a] = resume->u[a]; c[a] = resume->c[a]; }
    } else {
        /* O3 emit: frequency through the source CDF, isotropic direction */
        orc_uniforms(R->seed, pid, d++, R->pass, z);
        if (R->o->source_strata) {
            /* Eq. 1: the source spectrum is split into equal-energy bins with the same number
             * of packets each -- stratified sampling of the cumulative spectrum: packet pid takes stratum
             * pid mod S and a uniform position inside it */
            double S = (double)R->o->source_strata;
            z[0] = ((double)(pid % R->o->source_strata) + z[0]) / S;
        }
        j = orc_lower_bound(C->srccdf, nf, z[0]);
        orc_uniforms(R->seed, pid, d++, R->pass, z);
        orc_isotropic(z[0], z[1], u);
        p[0] = C->pos[0]; p[1] = C->pos[1]; p[2] = C->pos[2];
        start_cell(p, u, c);
        if (subR) {     /* the same rule on the lattice of sub-cube faces: cube and sub-cube of the start point */
            for (int a = 0; a < 3; ++a) {
                double pf = p[a] * (double)subR, fl = floor(pf);
                int G = (pf != fl) ? (int)fl : ((u[a] >= 0.0) ? (int)fl : (int)fl - 1);
                c[a] = (G >= 0) ? G / subR : -((-G + subR - 1) / subR);
                g[a] = G - c[a] * subR;
            }
            g_ok = 1;
        }
        hash_mix(&hash, event_word(ORC_EV_EMIT, j, ((uint64_t)c[2] * n[1] + c[1]) * n[0] + c[0]));
        st->packets++;
    }

    for (;;) { /* one flight per iteration */
        /* O4 / S3: optical depth to the next interaction, tau = -ln zeta (Eq. 3;
         * one draw per flight, the form of footnote 1; readings Q4-Q6) */
        orc_uniforms(R->seed, pid, d++, R->pass, z);
        double tau = -orc_det_log(z[0]);
        double ztype = z[1];
        st->flights++;
        orc_dda D;
        dda_setup(&D, p, u, c);
        double t = 0.0;
        size_t ci;
        int s, sj;
        double rho_c, kk;
        int first_cell = 1;
        int in_sub = 0;         /* the flight ends with an interaction inside sub-cube g */
        for (;;) {
            int blk = subR ? C->sub_of_cell[((size_t)c[2] * n[1] + c[1]) * n[0] + c[0]] : -1;
            if (blk < 0) g_ok = 0;
            else {
                /* a refined cube: the same walk on the lattice of its sub-cube faces, f = c + k/R (reading Q40) */
                const double Rd = (double)subR;
                if (!g_ok) {    /* entered from an unrefined cube: the sub-cube that holds the entry point p + u t.  Along the
                                 * crossed axis the point lies on the cube's face up to rounding, and the clamp makes that the
                                 * first or the last layer */
                    for (int a = 0; a < 3; ++a) {
                        double e = p[a] + u[a] * t;
                        int q = (int)floor((e - (double)c[a]) * Rd);
                        g[a] = q < 0 ? 0 : (q > subR - 1 ? subR - 1 : q);
                    }
                    g_ok = 1;
                }
                double ftm[3];
                for (int a = 0; a < 3; ++a)
                    ftm[a] = (D.step[a] == 0) ? INFINITY
                                              : (((double)c[a] + (double)(g[a] + (D.step[a] > 0 ? 1 : 0)) / Rd) - D.p[a]) * D.inv[a];
                int left = 0;
                while (!left) {
                    int a = (ftm[0] <= ftm[1] && ftm[0] <= ftm[2]) ? 0 : ((ftm[1] <= ftm[2]) ? 1 : 2);
                    double tn = ftm[a];
                    double ds = tn - t;
                    ci = nc0 + (size_t)blk * R3 + ((size_t)g[2] * subR + g[1]) * subR + g[0];
                    rho_c = (double)C->sub_rho[ci - nc0];
                    s = C->sub_sp[ci - nc0];
                    sj = s * nf + j;
                    if (R->o->per_cell_redraw && !first_cell) {
                        orc_uniforms(R->seed, pid, d++, R->pass, z);
                        tau = -orc_det_log(z[0]);
                    }
                    first_cell = 0;
                    kk = C->kext_h[sj] * rho_c;
                    double dtau = kk * ds;
                    if (dtau > tau) { in_sub = 1; break; }
                    tau -= dtau;
                    lucy_add(R, ci, sj, rho_c, ds, st);
                    t = tn;
                    g[a] += D.step[a];
                    ncross++;
                    st->crossings++;
                    if (rho_c > 0.0) st->dusty_crossings++;
                    if (g[a] < 0 || g[a] >= subR) {     /* through a face of the cube: the neighbouring cube, same sub-cube row */
                        g[a] = (D.step[a] > 0) ? 0 : subR - 1;
                        dda_advance(&D, a, c);
                        if (c[a] < 0 || c[a] >= n[a]) goto escaped;
                        left = 1;
                    } else {
                        ftm[a] = (((double)c[a] + (double)(g[a] + (D.step[a] > 0 ? 1 : 0)) / Rd) - D.p[a]) * D.inv[a];
                    }
                }
                if (in_sub) break;
                continue;
            }
            int a = dda_axis(&D);
            double tn = D.tmax[a];
            double ds = tn - t;
            ci = ((size_t)c[2] * n[1] + c[1]) * n[0] + c[0];
            rho_c = (double)C->rho[ci];
            s = C->sp[ci];
            sj = s * nf + j;
            if (R->o->per_cell_redraw && !first_cell) { /* new random number on cell entry */
                orc_uniforms(R->seed, pid, d++, R->pass, z);
                tau = -orc_det_log(z[0]);
            }
            first_cell = 0;
            kk = C->kext_h[sj] * rho_c;   /* Eq. 2 per unit path: (kabs+ksca) * h * rho */
            double dtau = kk * ds;        /* tau_i, Eq. 2 */
            if (dtau > tau) break;        /* interact inside this cell (reading Q5: equality leaves) */
            tau -= dtau;
            lucy_add(R, ci, sj, rho_c, ds, st);
            t = tn;
            dda_advance(&D, a, c);
            ncross++;
            st->crossings++;
            if (rho_c > 0.0) st->dusty_crossings++;
            if (c[a] < 0 || c[a] >= n[a]) goto escaped;
        }
        /* O5 interaction point: l' = tau / (rho (kabs+ksca)) (Eq. 3) */
        {
            double sint = tau / kk;
            lucy_add(R, ci, sj, rho_c, sint, st);
            double tint = t + sint;
            for (int a = 0; a < 3; ++a) {
                double q = p[a] + u[a] * tint;
                double lo = (double)c[a], hi = (double)(c[a] + 1);
                if (in_sub) {   /* the interaction point stays inside its sub-cube */
                    lo = (double)c[a] + (double)g[a] / (double)subR;
                    hi = (double)c[a] + (double)(g[a] + 1) / (double)subR;
                }
                if (q < lo) q = lo;
                if (q > hi) q = hi;
                p[a] = q;
            }
        }
        /* O6 scatter with probability albedo */
        if (ztype < C->albedo[sj]) {
            orc_uniforms(R->seed, pid, d++, R->pass, z);
            double un[3];
            /* (a mixture: the component that scatters, reading Q35) */
            const int cs = (comp_count(C, s) == 2 && !(ztype < C->mx_S0[sj])) ? 1 : 0;
            orc_hg_scatter(C->g[comp_mat(C, s, cs) * nf + j], z[0], z[1], u, un);
            if (R->sca_slot && R->sca_slot[j] >= 0) {   /* store the event: cell, frequency, incoming direction */
                uint64_t at = __atomic_fetch_add(R->sca_n, (uint64_t)1, __ATOMIC_RELAXED);
                if (at < R->sca_cap) {
                    orc_sca_event *ev = &R->sca_ev[at];
                    ev->cell = (uint32_t)ci; ev->slot = (uint16_t)R->sca_slot[j];
                    for (int a = 0; a < 3; ++a) ev->q[a] = (int16_t)llrint(32767.0 * u[a]);
                }
            }
            u[0] = un[0]; u[1] = un[1]; u[2] = un[2];
            nsca++;
            st->scatterings++;
            hash_mix(&hash, event_word(ORC_EV_SCATTER, j, ci));
        } else {
            /* O8 absorption: count it, re-emit at once from the same position with a new
             * frequency and an isotropic direction (readings Q18, Q20) */
            /* (a mixture: the component that absorbs, reading Q35; its count, temperature and emission row, Q36) */
            const int ca = (comp_count(C, s) == 2 && !(ztype < C->mx_A0[sj])) ? 1 : 0;
            __atomic_fetch_add(ca ? &R->k1[ci] : &R->k[ci], (uint64_t)1, __ATOMIC_RELAXED);
            nabs++;
            st->absorptions++;
            if (R->o->absorb_and_stop) {
                hash_mix(&hash, event_word(ORC_EV_ABSORB, j, ci));
                goto done;
            }
            int m = ca ? R->tidx1[ci] : R->tidx[ci];
            orc_uniforms(R->seed, pid, d++, R->pass, z);
            j = orc_lower_bound(R->cdf + ((size_t)comp_mat(C, s, ca) * C->nT + m) * nf, nf, z[0]); /* Eq. 10 / Eq. 5 */
            orc_uniforms(R->seed, pid, d++, R->pass, z);
            orc_isotropic(z[0], z[1], u);
            hash_mix(&hash, event_word(ORC_EV_ABSORB, j, ci));
        }
        /* carry-over (see orc_carry): the budget of this epoch is used up */
        if (R->carry_K && ++nint >= R->carry_K) {
            park->pid = pid; park->hash = hash; park->j = j; park->d = d;
            park->ncross = ncross; park->nsca = nsca; park->nabs = nabs;
            for (int a = 0; a < 3; ++a) { park->p[a] = p[a]; park->u[a] = u[a]; park->c[a] = c[a]; }
            return 1;
        }
    }
escaped:
    {
        /* O10 escape tally: frequency x |cos i| bin */
        double amu = fabs(u[2]);
        int bin = 0;
        for (int b = 1; b < C->ndir; ++b) if (C->mu_edges[b] <= amu) bin = b;
        __atomic_fetch_add(&R->sed[(size_t)bin * nf + j], (uint64_t)1, __ATOMIC_RELAXED);
        st->escapes++;
        if (nsca + nabs == 0) {
            __atomic_fetch_add(&R->sed_direct[(size_t)bin * nf + j], (uint64_t)1, __ATOMIC_RELAXED);
            st->direct_escapes++;
        }
        hash_mix(&hash, event_word(ORC_EV_ESCAPE, j, (uint64_t)bin));
        if (R->dig) R->dig[pid - R->pid0_digest].escape_bin = (uint32_t)bin;
    }
done:
    hash_mix(&hash, (uint64_t)ncross);
    hash_mix(&hash, (uint64_t)nsca | ((uint64_t)nabs << 32));
    if (R->dig) {
        orc_digest *g = &R->dig[pid - R->pid0_digest];
        g->hash = hash; g->crossings = ncross; g->scatterings = nsca; g->absorptions = nabs;
    }
    return 0;
}

/* growing list of carried packets */
typedef struct { orc_carry *v; size_t n, cap; } orc_carry_list;

static void carry_push(orc_carry_list *L, const orc_carry *e)
{
    if (L->n == L->cap) {
        L->cap = L->cap ? 2 * L->cap : 256;
        L->v = (orc_carry *)realloc(L->v, L->cap * sizeof(orc_carry));
    }
    L->v[L->n++] = *e;
}

static int carry_cmp(const void *a, const void *b)
{
    const uint64_t x = ((const orc_carry *)a)->pid, y = ((const orc_carry *)b)->pid;
    return x < y ? -1 : (x > y ? 1 : 0);
}

static void add_stats(orc_stats *total, const orc_stats *st)
{
    total->packets += st->packets; total->crossings += st->crossings;
    total->dusty_crossings += st->dusty_crossings; total->flights += st->flights;
    total->scatterings += st->scatterings; total->absorptions += st->absorptions;
    total->escapes += st->escapes; total->direct_escapes += st->direct_escapes;
    total->lucy_adds += st->lucy_adds;
}

/* One epoch's packets: first the packets carried over from the previous epoch (`in`), then `count` new packets
 * with ids from pid0.  Packets whose budget runs out are appended to `out` (sorted by id afterwards, so that the
 * list does not depend on the thread count). */
static void run_range(orc_run_t *R, uint64_t pid0, uint64_t count, orc_stats *total, const orc_carry_list *in,
                      orc_carry_list *out)
{
    int nth = R->o->n_threads > 1 ? R->o->n_threads : 1;
    if (R->Lsum) nth = 1;
    const int64_t n_in = in ? (int64_t)in->n : 0, n_all = n_in + (int64_t)count;
#ifdef _OPENMP
    if (nth > 1) {
        /* packets are independent inside an epoch; integer tallies make the result
         * independent of the thread count */
#pragma omp parallel num_threads(nth)
        {
            orc_stats st;
            memset(&st, 0, sizeof st);
            orc_carry_list mine = { NULL, 0, 0 };
            orc_carry e;
#pragma omp for schedule(dynamic, 64)
            for (int64_t i = 0; i < n_all; ++i) {
                const int parked = (i < n_in) ? run_packet(R, 0, &st, &in->v[i], &e)
                                              : run_packet(R, pid0 + (uint64_t)(i - n_in), &st, NULL, &e);
                if (parked) carry_push(&mine, &e);
            }
#pragma omp critical
            {
                add_stats(total, &st);
                for (size_t q = 0; q < mine.n; ++q) carry_push(out, &mine.v[q]);
            }
            free(mine.v);
        }
        if (out && out->n > 1) qsort(out->v, out->n, sizeof(orc_carry), carry_cmp);
        return;
    }
#endif
    orc_carry e;
    for (int64_t i = 0; i < n_all; ++i) {
        const int parked = (i < n_in) ? run_packet(R, 0, total, &in->v[i], &e)
                                      : run_packet(R, pid0 + (uint64_t)(i - n_in), total, NULL, &e);
        if (parked) carry_push(out, &e);
    }
    if (out && out->n > 1) qsort(out->v, out->n, sizeof(orc_carry), carry_cmp);
}

/* number of J[s][.] entries strictly below x, clamped to [0, nT-1] */
static inline int t_index(const orc_ctx *C, int s, double x)
{
    const double *J = C->J + (size_t)s * C->nT;
    int lo = 0, hi = C->nT; /* first index with J >= x */
    while (lo < hi) {
        int mid = (lo + hi) / 2;
        if (J[mid] < x) lo = mid + 1; else hi = mid;
    }
    if (lo > C->nT - 1) lo = C->nT - 1;
    return lo;
}

typedef struct {
    const orc_ctx *C;
    size_t nc;
    uint64_t *k, *kprev;
    int64_t *Lfx;
    double *Lsum, *Lcmp;
    uint16_t *tidx;
    uint64_t *k1, *kprev1;   /* second component of a mixture (NEXT-3); NULL without mixtures */
    int64_t *Lfx1;
    uint16_t *tidx1;
    uint64_t *sed, *sed_direct;
    int fx;
    int hybrid;              /* the stored tallies were made with lucy_hybrid */
    double *kmax_diag;       /* [ns] sqrt(3) h max_nu (kabs + ksca), reading Q37 */
    double xi;               /* packet energy L/N of the run that produced the stored tallies */
    int32_t *sca_slot;       /* [nf] slot of a recorded frequency bin, -1 otherwise; NULL = nothing is recorded */
    int n_sca_bins;
    int32_t sca_bins[16];
    orc_sca_event *sca_ev;
    uint64_t sca_cap, sca_n;
} orc_state;

orc_state *orc_state_create(const orc_ctx *C)
{
    orc_state *S = (orc_state *)calloc(1, sizeof(orc_state));
    S->C = C;
    S->nc = cells_total(C);          /* sub-cubes (NEXT-3) are cells of their own, behind the grid's */
    S->k = (uint64_t *)calloc(S->nc, sizeof(uint64_t));
    S->kprev = (uint64_t *)calloc(S->nc, sizeof(uint64_t));
    S->Lfx = (int64_t *)calloc(S->nc, sizeof(int64_t));
    S->tidx = (uint16_t *)calloc(S->nc, sizeof(uint16_t));
    if (C->n_mix) {
        S->k1 = (uint64_t *)calloc(S->nc, sizeof(uint64_t));
        S->kprev1 = (uint64_t *)calloc(S->nc, sizeof(uint64_t));
        S->Lfx1 = (int64_t *)calloc(S->nc, sizeof(int64_t));
        S->tidx1 = (uint16_t *)calloc(S->nc, sizeof(uint16_t));
    }
    S->sed = (uint64_t *)calloc((size_t)C->ndir * C->nf, sizeof(uint64_t));
    S->sed_direct = (uint64_t *)calloc((size_t)C->ndir * C->nf, sizeof(uint64_t));
    return S;
}

void orc_state_destroy(orc_state *S)
{
    if (!S) return;
    free(S->k); free(S->kprev); free(S->Lfx); free(S->Lsum); free(S->Lcmp); free(S->tidx);
    free(S->k1); free(S->kprev1); free(S->Lfx1); free(S->tidx1); free(S->kmax_diag);
    free(S->sed); free(S->sed_direct); free(S->sca_slot); free(S->sca_ev); free(S);
}

static void zero_tallies(orc_state *S)
{
    memset(S->k, 0, S->nc * sizeof(uint64_t));
    memset(S->kprev, 0, S->nc * sizeof(uint64_t));
    memset(S->Lfx, 0, S->nc * sizeof(int64_t));
    if (S->k1) {
        memset(S->k1, 0, S->nc * sizeof(uint64_t));
        memset(S->kprev1, 0, S->nc * sizeof(uint64_t));
        memset(S->Lfx1, 0, S->nc * sizeof(int64_t));
    }
    if (S->Lsum) { memset(S->Lsum, 0, S->nc * sizeof(double)); memset(S->Lcmp, 0, S->nc * sizeof(double)); }
    memset(S->sed, 0, (size_t)S->C->ndir * S->C->nf * sizeof(uint64_t));
    memset(S->sed_direct, 0, (size_t)S->C->ndir * S->C->nf * sizeof(uint64_t));
    S->sca_n = 0;
}

/* fixed-point fraction bits (O9): FX = min(40, 58 - ceil(log2 N)) */
int orc_fx_bits(uint64_t n_packets)
{
    int cl = 0;
    while (((uint64_t)1 << cl) < n_packets && cl < 63) ++cl;
    int fx = 58 - cl;
    if (fx > 40) fx = 40;
    if (fx < 0) fx = 0;
    return fx;
}

/* default epoch schedule (O11, reading Q19): B0 = max(256, largest power of two <= N/256), Bmax = 2^22 */
void orc_default_schedule(uint64_t n_packets, uint64_t *B0, uint64_t *Bmax)
{
    uint64_t q = n_packets / 256, b = 256;
    while (b * 2 <= q) b *= 2;
    *B0 = b;
    *Bmax = (uint64_t)1 << 22;
}

/* O11 epoch rule.  Bjorkman & Wood adjust the temperature after every absorption;
 * under parallel execution the order of absorptions is undefined, so packets are
 * processed in epochs in pid order and the temperature index of every cell is frozen inside an epoch
 * at a midpoint prediction of its count (reading Q19/Q20):
 *   k~ = k + max(1, 1/2 (k - k_prev) B_e / B_{e-1}),   x = k~ xi / (4 pi rho h^3)   (Eq. 4)
 *   tidx = #{ J[s][.] < x } clamped. */
static void epoch_update(orc_state *S, int first_epoch, double ratio, double cellfac)
{
    const orc_ctx *C = S->C;
    const double inv_fx = ldexp(1.0, -S->fx);
    const size_t nc0 = (size_t)C->nx * C->ny * C->nz;
    const double cellfac0 = cellfac, cellfac_sub = cellfac * (double)(C->subR * C->subR * C->subR);   /* V = (h/R)^3 */
    for (size_t ci = 0; ci < S->nc; ++ci) {
        double rho_c = cell_rho(C, ci);
        uint64_t kk = S->k[ci];
        if (ci >= nc0) cellfac = cellfac_sub; else cellfac = cellfac0;
        if (ci >= nc0 || (C->subR && C->sub_of_cell[ci] >= 0)) {      /* a sub-cube, or a refined cube (no dust of its own) */
            if (rho_c > 0.0) {
                double kt;
                if (first_epoch) kt = (double)kk + 1.0;
                else {
                    double pred = 0.5 * (double)(kk - S->kprev[ci]) * ratio;
                    kt = (double)kk + ((pred > 1.0) ? pred : 1.0);
                }
                S->tidx[ci] = (uint16_t)t_index(C, cell_sp(C, ci), kt * cellfac / rho_c);
            } else S->tidx[ci] = 0;
            S->kprev[ci] = kk;
            continue;
        }
        if (S->hybrid && orc_thin_cell(rho_c, S->kmax_diag[C->sp[ci]])) {
            /* Sect. 3.1 (reading Q39): the temperature of a cell below the threshold comes from its Eq. 9 energy, Eq. 4
             * with k xi replaced by E_abs; the same midpoint prediction, on the tally (k_prev keeps the tally here) */
            double E = (double)S->Lfx[ci] * inv_fx, Ep = (double)(int64_t)S->kprev[ci] * inv_fx;
            double Et = first_epoch ? E : E + 0.5 * (E - Ep) * ratio;
            S->tidx[ci] = (uint16_t)t_index(C, C->sp[ci], Et * cellfac / rho_c);
            S->kprev[ci] = (uint64_t)S->Lfx[ci];
            continue;
        }
        if (rho_c > 0.0) {
            double kt;
            if (first_epoch) kt = (double)kk + 1.0;
            else {
                double pred = 0.5 * (double)(kk - S->kprev[ci]) * ratio;
                kt = (double)kk + ((pred > 1.0) ? pred : 1.0);
            }
            /* (a mixture: Eq. 4 with the component's own mass rho f_c V, reading Q36) */
            double x = kt * cellfac / (C->n_mix ? rho_c * C->mx_frac[2 * C->sp[ci]] : rho_c);
            S->tidx[ci] = (uint16_t)t_index(C, comp_mat(C, C->sp[ci], 0), x);
        } else {
            S->tidx[ci] = 0;
        }
        S->kprev[ci] = kk;
        if (S->k1) {    /* the second component: the same rule on its own count */
            const int xm = C->sp[ci];
            uint64_t k1 = S->k1[ci];
            if (rho_c > 0.0 && C->mx_ncomp[xm] == 2) {
                double kt;
                if (first_epoch) kt = (double)k1 + 1.0;
                else {
                    double pred = 0.5 * (double)(k1 - S->kprev1[ci]) * ratio;
                    kt = (double)k1 + ((pred > 1.0) ? pred : 1.0);
                }
                double x = kt * cellfac / (rho_c * C->mx_frac[2 * xm + 1]);
                S->tidx1[ci] = (uint16_t)t_index(C, C->mx_mat[2 * xm + 1], x);
            } else {
                S->tidx1[ci] = 0;
            }
            S->kprev1[ci] = k1;
        }
    }
}

/* S12: temperature index for a frozen-T sweep from the previous pass's tallies */
static void sweep_update(orc_state *S, int from_lucy, double cellfac, int fx_of_tallies)
{
    const orc_ctx *C = S->C;
    double inv_fx = ldexp(1.0, -fx_of_tallies);
    const size_t nc0 = (size_t)C->nx * C->ny * C->nz;
    const double cellfac_sub = cellfac * (double)(C->subR * C->subR * C->subR);
    for (size_t ci = 0; ci < S->nc; ++ci) {
        double rho_c = cell_rho(C, ci);
        if (ci >= nc0 || (C->subR && C->sub_of_cell[ci] >= 0)) {
            if (rho_c > 0.0) {
                double e = from_lucy ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
                S->tidx[ci] = (uint16_t)t_index(C, cell_sp(C, ci), e * (ci >= nc0 ? cellfac_sub : cellfac) / rho_c);
            } else S->tidx[ci] = 0;
            continue;
        }
        if (rho_c > 0.0) {
            double e = from_lucy ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
            if (S->hybrid) e = orc_thin_cell(rho_c, S->kmax_diag[C->sp[ci]]) ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
            double x = e * cellfac / (C->n_mix ? rho_c * C->mx_frac[2 * C->sp[ci]] : rho_c);
            S->tidx[ci] = (uint16_t)t_index(C, comp_mat(C, C->sp[ci], 0), x);
        } else {
            S->tidx[ci] = 0;
        }
        if (S->k1) {
            const int xm = C->sp[ci];
            if (rho_c > 0.0 && C->mx_ncomp[xm] == 2) {
                double e = from_lucy ? (double)S->Lfx1[ci] * inv_fx : (double)S->k1[ci];
                double x = e * cellfac / (rho_c * C->mx_frac[2 * xm + 1]);
                S->tidx1[ci] = (uint16_t)t_index(C, C->mx_mat[2 * xm + 1], x);
            } else {
                S->tidx1[ci] = 0;
            }
        }
    }
}

/* O-run: the whole path for N packets.  Returns 0, -5 on fixed-point overflow (|L| > 2^62), -2 when a run
 * without reset would mix tallies of different packet energies. */
int orc_run(orc_state *S, uint64_t n_packets, uint64_t seed, const orc_opts *o, orc_stats *stats,
            orc_digest *digests)
{
    const orc_ctx *C = S->C;
    orc_stats st;
    memset(&st, 0, sizeof st);
    orc_run_t R;
    memset(&R, 0, sizeof R);
    if (o->keep_fp64_lucy && !S->Lsum) {
        S->Lsum = (double *)calloc(S->nc, sizeof(double));
        S->Lcmp = (double *)calloc(S->nc, sizeof(double));
    }
    /* sweeps (S12) take their temperatures from the previous pass's tallies, so only a B&W run resets first */
    if (o->reset && o->mode == ORC_MODE_BW_EPOCH) zero_tallies(S);
    const uint64_t n_xi = o->n_total ? o->n_total : n_packets;
    /* the stored tallies are in units of the packet energy and fixed-point scale of the run that made them */
    const int prev_fx = S->fx;
    const double prev_xi = S->xi;
    S->fx = orc_fx_bits(n_xi);
    S->xi = C->L / (double)n_xi;                         /* xi = L/N */
    if (!o->reset && o->mode == ORC_MODE_BW_EPOCH && prev_xi != 0.0 && (prev_xi != S->xi || prev_fx != S->fx))
        return -2;                                       /* tallies of another packet energy cannot be continued */
    if (o->lucy_hybrid && (C->n_mix || C->subR)) return -3; /* not defined for mixtures / sub-cubes */
    if (C->subR && o->carry_K) return -3;
    if (!o->reset && prev_xi != 0.0 && (S->hybrid != 0) != (o->lucy_hybrid != 0))
        return -2;                                       /* tallies of the other estimator cannot be continued */
    if (o->lucy_hybrid && !S->kmax_diag) {
        S->kmax_diag = (double *)malloc(C->ns * sizeof(double));
        for (int s = 0; s < C->ns; ++s) {
            double km = 0.0;
            for (int j = 0; j < C->nf; ++j) {
                double ke = C->kabs[s * C->nf + j] + C->ksca[s * C->nf + j];
                if (ke > km) km = ke;
            }
            S->kmax_diag[s] = sqrt(3.0) * C->h * km;
        }
    }
    S->hybrid = o->lucy_hybrid ? 1 : 0;
    double cellfac = S->xi / (ORC_FOUR_PI * C->h * C->h * C->h); /* xi / (4 pi V), Eq. 4 */
    /* Eq. 4 for the first sweep: k and L were counted in packets of the PREVIOUS run's energy */
    double prev_cellfac = prev_xi / (ORC_FOUR_PI * C->h * C->h * C->h);
    size_t nsf = (size_t)C->ntab * C->nf;
    R.C = C; R.k = S->k; R.kprev = S->kprev; R.Lfx = S->Lfx; R.tidx = S->tidx;
    R.k1 = S->k1; R.Lfx1 = S->Lfx1; R.tidx1 = S->tidx1;
    R.kmax_diag = S->hybrid ? S->kmax_diag : NULL;
    R.Lsum = o->keep_fp64_lucy ? S->Lsum : NULL; R.Lcmp = S->Lcmp;
    R.sed = S->sed; R.sed_direct = S->sed_direct; R.dig = digests; R.seed = seed; R.fx = S->fx; R.o = o;
    R.pid0_digest = o->pid0;
    R.sca_slot = S->sca_slot; R.sca_ev = S->sca_ev; R.sca_cap = S->sca_cap; R.sca_n = &S->sca_n;
    R.kabs_fx = (double *)malloc(nsf * sizeof(double));
    for (size_t i = 0; i < nsf; ++i) R.kabs_fx[i] = ldexp(C->kabs_h[i], S->fx);
    if (C->n_mix) {
        R.kabs1_fx = (double *)malloc(nsf * sizeof(double));
        for (size_t i = 0; i < nsf; ++i) R.kabs1_fx[i] = ldexp(C->mx_kabs1_h[i], S->fx);
    }
    st.fx_bits = S->fx;

    if (o->mode == ORC_MODE_BW_EPOCH) {
        uint64_t B0 = o->B0, Bmax = o->Bmax, d0, d1;
        orc_default_schedule(n_packets, &d0, &d1);
        if (B0 == 0) B0 = d0;
        if (Bmax == 0) Bmax = d1;
        if (Bmax < B0) Bmax = B0;
        R.cdf = C->cdfdB;
        R.pass = o->pass0;
        uint64_t done = 0, Bnom = B0, Bprev = 0;
        int e = 0;
        orc_carry_list carried = { NULL, 0, 0 }, parked = { NULL, 0, 0 };
        R.carry_K = o->absorb_and_stop ? 0u : o->carry_K;
        while (done < n_packets) {
            uint64_t Be = n_packets - done < Bnom ? n_packets - done : Bnom;
            epoch_update(S, e == 0, e == 0 ? 1.0 : (double)Be / (double)Bprev, cellfac);
            parked.n = 0;
            run_range(&R, o->pid0 + done, Be, &st, &carried, &parked);
            { orc_carry_list t = carried; carried = parked; parked = t; }
            done += Be;
            Bprev = Be;
            {
                double nb = floor((double)Bnom * (o->growth > 0.0 ? o->growth : 2.0));
                uint64_t nn = nb >= 1.8e19 ? Bmax : (uint64_t)nb;
                if (nn < Bnom) nn = Bnom;
                Bnom = nn > Bmax ? Bmax : nn;
            }
            ++e;
            st.epochs++;
        }
        /* the packets still carried run in further epochs (no new packets, same temperature rule with B_e / B_e-1
         * = 1), the budget doubling each time, until all have escaped */
        while (carried.n > 0) {
            R.carry_K = R.carry_K > 0x40000000u ? 0x80000000u : 2u * R.carry_K;
            epoch_update(S, 0, 1.0, cellfac);
            parked.n = 0;
            run_range(&R, 0, 0, &st, &carried, &parked);
            { orc_carry_list t = carried; carried = parked; parked = t; }
            st.epochs++;
        }
        free(carried.v); free(parked.v);
    } else {
        /* iterative scheme of PAPER.md:73: temperatures of the previous run, Eq. 5 for the frequency */
        R.cdf = C->cdfB;
        for (int sw = 1; sw <= o->n_sweeps; ++sw) {
            /* counters describe the tallies they go with: each sweep starts both from zero */
            uint64_t ep = st.epochs;
            memset(&st, 0, sizeof st);
            st.epochs = ep;
            st.fx_bits = S->fx;
            sweep_update(S, o->sweep_T_from_lucy, sw == 1 ? prev_cellfac : cellfac, sw == 1 ? prev_fx : S->fx);
            zero_tallies(S);
            R.pass = o->pass0 + (uint32_t)sw;
            R.carry_K = 0;
            run_range(&R, o->pid0, n_packets, &st, NULL, NULL);
            st.epochs++;
        }
    }
    free(R.kabs_fx); free(R.kabs1_fx);
    for (size_t ci = 0; ci < S->nc; ++ci) {
        int64_t v = S->Lfx[ci];
        if (v > ((int64_t)1 << 62) || v < -((int64_t)1 << 62)) st.overflow = 1;
        if (S->Lfx1) {
            v = S->Lfx1[ci];
            if (v > ((int64_t)1 << 62) || v < -((int64_t)1 << 62)) st.overflow = 1;
        }
    }
    if (stats) *stats = st;
    return st.overflow ? -5 : 0;
}

/* raw tallies for the parity tests */
void orc_read_raw(const orc_state *S, uint64_t *k, int64_t *Lfx, uint64_t *sed, uint64_t *sed_direct,
                  uint16_t *tidx, double *Lsum)
{
    if (k) memcpy(k, S->k, S->nc * sizeof(uint64_t));
    if (Lfx) memcpy(Lfx, S->Lfx, S->nc * sizeof(int64_t));
    if (sed) memcpy(sed, S->sed, (size_t)S->C->ndir * S->C->nf * sizeof(uint64_t));
    if (sed_direct) memcpy(sed_direct, S->sed_direct, (size_t)S->C->ndir * S->C->nf * sizeof(uint64_t));
    if (tidx) memcpy(tidx, S->tidx, S->nc * sizeof(uint16_t));
    if (Lsum && S->Lsum) memcpy(Lsum, S->Lsum, S->nc * sizeof(double));
}

/* Eq. 9 as evaluated by lucy_add, for the pin that compares it with 1 - exp(-tau) */
double orc_eq9_value(double tau) { return orc_eq9(tau); }

/* raw tallies of the second component of a mixture (NEXT-3) */
int orc_read_raw_comp1(const orc_state *S, uint64_t *k, int64_t *Lfx, uint16_t *tidx)
{
    if (!S->k1) return -1;
    if (k) memcpy(k, S->k1, S->nc * sizeof(uint64_t));
    if (Lfx) memcpy(Lfx, S->Lfx1, S->nc * sizeof(int64_t));
    if (tidx) memcpy(tidx, S->tidx1, S->nc * sizeof(uint16_t));
    return 0;
}

/* invert J[s](T) = x by log-log interpolation (O12; Eq. 4; clamp per reading Q16) */
double orc_T_of_x(const orc_ctx *C, int s, double x)
{
    const double *J = C->J + (size_t)s * C->nT;
    if (!(x > 0.0)) return 0.0;
    if (x <= J[0]) return C->Tg[0];
    if (x >= J[C->nT - 1]) return C->Tg[C->nT - 1];
    int lo = 0, hi = C->nT - 1; /* J[lo] <= x < J[hi] */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (J[mid] <= x) lo = mid; else hi = mid;
    }
    double f = log(x / J[lo]) / log(J[hi] / J[lo]);
    return C->Tg[lo] * exp(f * log(C->Tg[hi] / C->Tg[lo]));
}

/* O12 physical outputs: E_count = k xi, E_lucy = xi L / 2^FX (erg/s absorbed per cell), T from either,
 * SED = counts xi / (dnu_j dOmega_bin), dOmega_bin = 4 pi d|mu| (both hemispheres; reading Q22). */
void orc_read(const orc_state *S, double *E_count, double *E_lucy, float *T, int T_from_lucy, double *SED)
{
    const orc_ctx *C = S->C;
    double inv_fx = ldexp(1.0, -S->fx);
    double cellfac = S->xi / (ORC_FOUR_PI * C->h * C->h * C->h);
    for (size_t ci = 0; ci < S->nc; ++ci) {
        double ec = (double)S->k[ci] * S->xi;
        double el = (double)S->Lfx[ci] * inv_fx * S->xi;
        if (E_count) E_count[ci] = ec;
        if (E_lucy) E_lucy[ci] = el;
        if (T && C->subR) {          /* grids with sub-cubes: every cell with its own volume */
            double rho_c = cell_rho(C, ci);
            double e = T_from_lucy ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
            T[ci] = rho_c > 0.0 ? (float)orc_T_of_x(C, cell_sp(C, ci), e * cell_fac(C, ci, S->xi) / rho_c) : 0.0f;
        } else if (T) {
            double rho_c = (double)C->rho[ci];
            if (rho_c > 0.0) {
                double e = T_from_lucy ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
                if (T_from_lucy == 2)   /* Sect. 3.1: Eq. 9 energy below the threshold, counts above (reading Q39) */
                    e = (S->kmax_diag && orc_thin_cell(rho_c, S->kmax_diag[C->sp[ci]])) ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
                double mass = C->n_mix ? rho_c * C->mx_frac[2 * C->sp[ci]] : rho_c;
                T[ci] = (float)orc_T_of_x(C, comp_mat(C, C->sp[ci], 0), e * cellfac / mass);
            } else T[ci] = 0.0f;
        }
    }
    if (SED)
        for (int b = 0; b < C->ndir; ++b)
            for (int j = 0; j < C->nf; ++j) {
                double dom = ORC_FOUR_PI * (C->mu_edges[b + 1] - C->mu_edges[b]);
                SED[(size_t)b * C->nf + j] = (double)S->sed[(size_t)b * C->nf + j] * S->xi / (C->dnu[j] * dom);
            }
}

/* the same outputs for the second component of a mixture (NEXT-3, reading Q36): energy absorbed by that component and
 * its temperature (0 in cells whose mixture has one component) */
int orc_read_comp1(const orc_state *S, double *E_count, double *E_lucy, float *T, int T_from_lucy)
{
    const orc_ctx *C = S->C;
    if (!S->k1) return -1;
    double inv_fx = ldexp(1.0, -S->fx);
    double cellfac = S->xi / (ORC_FOUR_PI * C->h * C->h * C->h);
    for (size_t ci = 0; ci < S->nc; ++ci) {
        if (E_count) E_count[ci] = (double)S->k1[ci] * S->xi;
        if (E_lucy) E_lucy[ci] = (double)S->Lfx1[ci] * inv_fx * S->xi;
        if (T) {
            double rho_c = (double)C->rho[ci];
            const int xm = C->sp[ci];
            if (rho_c > 0.0 && C->mx_ncomp[xm] == 2) {
                double e = T_from_lucy ? (double)S->Lfx1[ci] * inv_fx : (double)S->k1[ci];
                T[ci] = (float)orc_T_of_x(C, C->mx_mat[2 * xm + 1], e * cellfac / (rho_c * C->mx_frac[2 * xm + 1]));
            } else T[ci] = 0.0f;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-2  Scattering-event store and ray tracer (Sect. 4, Eq. 11-17).
 * ---------------------------------------------------------------------------------------------- */
/* record the scattering events of later runs at these frequency bins (at most 16), up to `capacity` events */
int orc_scatter_store(orc_state *S, int n_bins, const int32_t *bins, uint64_t capacity)
{
    if (n_bins < 1 || n_bins > 16) return -1;
    free(S->sca_slot); free(S->sca_ev);
    S->sca_slot = (int32_t *)malloc(S->C->nf * sizeof(int32_t));
    for (int j = 0; j < S->C->nf; ++j) S->sca_slot[j] = -1;
    for (int b = 0; b < n_bins; ++b) {
        if (bins[b] < 0 || bins[b] >= S->C->nf) return -1;
        S->sca_slot[bins[b]] = b; S->sca_bins[b] = bins[b];
    }
    S->n_sca_bins = n_bins;
    S->sca_ev = (orc_sca_event *)malloc((capacity ? capacity : 1) * sizeof(orc_sca_event));
    S->sca_cap = capacity; S->sca_n = 0;
    return 0;
}

uint64_t orc_scatter_events(const orc_state *S, orc_sca_event *out, uint64_t max_n)
{
    uint64_t n = S->sca_n < S->sca_cap ? S->sca_n : S->sca_cap;
    if (out) memcpy(out, S->sca_ev, (size_t)(n < max_n ? n : max_n) * sizeof(orc_sca_event));
    return S->sca_n;
}

/* Henyey-Greenstein phase function, per steradian (Eq. 15) */
double orc_phase_hg(double g, double cos_beta)
{
    double d = 1.0 + g * g - 2.0 * g * cos_beta;
    return (1.0 - g * g) / (ORC_FOUR_PI * d * sqrt(d));
}

/* The image of Sect. 4 at frequency bin j for an observer in direction ez (unit vector from the object towards the
 * observer) at distance D, parallel projection (Eq. 11): pixel (a, b) of nx x ny pixels of size pix looks along the
 * line r = i0 + (a + 1/2 - nx/2) pix ex + (b + 1/2 - ny/2) pix ey + s ez, i0 = centre of the grid, ey = ez x ex.
 * Along the line, from the observer's side inwards, every cell i adds (Eq. 12, 17)
 *     A_pix / D^2 * (I_e + I_s) * exp(-tau),   tau = sum of the tau_cell of the cells between i and the observer,
 *     tau_cell = kappa_abs rho l (Eq. 13: absorption cross section, as printed), l = length of the line inside the cell,
 *     I_e = (1 - exp(-tau_cell)) B_nu(T_i)                                            (Eq. 14)
 *     I_s = l / V * sum over the cell's stored events of P_HG(beta) xi / dnu           (Eq. 16)
 * with beta the angle between ez and the event's incoming direction, V = h^3 (the events' scattered luminosity per
 * steradian towards the observer, spread over the cell's volume -- reading Q30: Eq. 16 gives no normalisation).
 * T_i inverts Eq. 4 from the counts (T_from_lucy = 0) or the Lucy tally (1).  Fe / Fs: [ny][nx], erg s^-1 cm^-2 Hz^-1. */
int orc_ray_trace(const orc_state *S, const double ez_in[3], const double ex_in[3], int nx, int ny, double pix, double D,
                  int j, int T_from_lucy, double *Fe, double *Fs)
{
    const orc_ctx *C = S->C;
    if (j < 0 || j >= C->nf || nx < 1 || ny < 1 || !(pix > 0.0) || !(D > 0.0)) return -1;
    if (C->n_mix || C->subR) return -1;    /* images of mixtures / refined grids are not defined here */
    const int n[3] = { C->nx, C->ny, C->nz };
    double ez[3], ex[3], ey[3];
    double nz_ = sqrt(ez_in[0] * ez_in[0] + ez_in[1] * ez_in[1] + ez_in[2] * ez_in[2]);
    for (int a = 0; a < 3; ++a) ez[a] = ez_in[a] / nz_;
    double dot = ex_in[0] * ez[0] + ex_in[1] * ez[1] + ex_in[2] * ez[2];
    for (int a = 0; a < 3; ++a) ex[a] = ex_in[a] - dot * ez[a];
    double nx_ = sqrt(ex[0] * ex[0] + ex[1] * ex[1] + ex[2] * ex[2]);
    if (!(nx_ > 0.0)) return -1;
    for (int a = 0; a < 3; ++a) ex[a] /= nx_;
    ey[0] = ez[1] * ex[2] - ez[2] * ex[1]; ey[1] = ez[2] * ex[0] - ez[0] * ex[2]; ey[2] = ez[0] * ex[1] - ez[1] * ex[0];
    /* per-cell sum of P_HG(beta) over the stored events of this frequency (the sum over beta of Eq. 16) */
    size_t nc = S->nc;
    double *src = (double *)calloc(nc, sizeof(double));
    int slot = (S->sca_slot) ? S->sca_slot[j] : -1;
    if (slot >= 0) {
        uint64_t ne = S->sca_n < S->sca_cap ? S->sca_n : S->sca_cap;
        for (uint64_t e = 0; e < ne; ++e) {
            const orc_sca_event *ev = &S->sca_ev[e];
            if (ev->slot != slot) continue;
            double qx = ev->q[0], qy = ev->q[1], qz = ev->q[2];
            double qn = sqrt(qx * qx + qy * qy + qz * qz);
            double cb = (qx * ez[0] + qy * ez[1] + qz * ez[2]) / qn;
            src[ev->cell] += orc_phase_hg(C->g[C->sp[ev->cell] * C->nf + j], cb);
        }
    }
    const double inv_fx = ldexp(1.0, -S->fx);
    const double cellfac = S->xi / (ORC_FOUR_PI * C->h * C->h * C->h);
    const double apix_d2 = pix * pix / (D * D);
    const double V = C->h * C->h * C->h;
    const double u[3] = { -ez[0], -ez[1], -ez[2] };     /* the walk runs from the observer's side inwards */
    for (int b = 0; b < ny; ++b)
        for (int a = 0; a < nx; ++a) {
            double fe = 0.0, fs = 0.0;
            /* point of the line in cell units, then the slab parameters at which it is inside the grid */
            double r0[3], smin = -INFINITY, smax = INFINITY;
            double xa = ((double)a + 0.5 - 0.5 * nx) * pix / C->h, yb = ((double)b + 0.5 - 0.5 * ny) * pix / C->h;
            for (int q = 0; q < 3; ++q) r0[q] = 0.5 * n[q] + xa * ex[q] + yb * ey[q];
            int miss = 0;
            for (int q = 0; q < 3; ++q) {
                if (u[q] == 0.0) { if (!(r0[q] > 0.0 && r0[q] < (double)n[q])) miss = 1; continue; }
                double s1 = (0.0 - r0[q]) / u[q], s2 = ((double)n[q] - r0[q]) / u[q];
                double lo = s1 < s2 ? s1 : s2, hi = s1 < s2 ? s2 : s1;
                if (lo > smin) smin = lo;
                if (hi < smax) smax = hi;
            }
            if (!miss && smax > smin) {
                double p[3];
                int c[3];
                for (int q = 0; q < 3; ++q) {
                    p[q] = r0[q] + smin * u[q];
                    if (p[q] < 0.0) p[q] = 0.0;
                    if (p[q] > (double)n[q]) p[q] = (double)n[q];
                }
                start_cell(p, u, c);
                int inside = 1;
                for (int q = 0; q < 3; ++q) if (c[q] < 0 || c[q] >= n[q]) inside = 0;
                if (inside) {
                    orc_dda Dd;
                    dda_setup(&Dd, p, u, c);
                    double t = 0.0, tau = 0.0;
                    for (;;) {
                        int ax = dda_axis(&Dd);
                        double tn = Dd.tmax[ax], l = (tn - t) * C->h;
                        size_t ci = ((size_t)c[2] * n[1] + c[1]) * n[0] + c[0];
                        double rho_c = (double)C->rho[ci];
                        if (rho_c > 0.0) {
                            int sp = C->sp[ci];
                            double tc = C->kabs[sp * C->nf + j] * rho_c * l;
                            double e = T_from_lucy ? (double)S->Lfx[ci] * inv_fx : (double)S->k[ci];
                            double T = orc_T_of_x(C, sp, e * cellfac / rho_c);
                            double att = exp(-tau);
                            if (T > 0.0) fe += -expm1(-tc) * orc_planck(C->nu[j], T) * att;
                            fs += l / V * src[ci] * S->xi / C->dnu[j] * att;
                            tau += tc;
                        }
                        t = tn;
                        dda_advance(&Dd, ax, c);
                        if (c[ax] < 0 || c[ax] >= n[ax]) break;
                    }
                }
            }
            Fe[(size_t)b * nx + a] = fe * apix_d2;
            if (Fs) Fs[(size_t)b * nx + a] = fs * apix_d2;
        }
    free(src);
    return 0;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
