/*
 * dies_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, serial, fp64 CPU implementation of the immediate re-emission (IRE) Monte Carlo
 * of DIES (arXiv 2408.13807) for a 1D spherical cloud of concentric shells, written from the
 * paper (/root/reference/PAPER.md, cited below as PAPER.md:L<line>) and from the readings listed
 * in DESIGN.md ("Readings of the paper", R1..R20).  One photon package is followed to the end
 * before the next one starts.  No blocking, no fusion, no reordering.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table generator or constant with the CUDA path
 * (paper_2408_13807_b200/csrc); the Philox4x32-10 generator is implemented here independently
 * from the written contract.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox4x32_10 ............ Random123 known-answer vectors (tests/golden/philox_kat.txt)
 *   shell stepping ........... brute-force 3-D line/sphere intersection (north_star check a)
 *   launch + geometry ........ kappa=0: mean path length in shell i = V_i/(pi R^2) (Cauchy), mean chord 4R/3
 *   first-flight extinction .. closed form 1-[1-(1+2t)e^{-2t}]/(2t^2) for a uniform sphere
 *   HG sampling .............. <cos Theta> = g, chi^2 against Eq. 6
 *   energy conservation ...... escaped = injected to 1e-9 (north_star check b)
 *   T lookup ................. T(eps_t) = T_t;  sum_i m_i eps(T_i) = absorbed energy
 *   re-emission .............. telescoping: re-emitted spectrum of a cell = C(eps_final); order independence
 *   optically thin limit ..... int kappa J = int kappa B(T) within 0.5 % (north_star check c)
 *   IRE vs iteration ......... agreement with an independent 3-D Cartesian TMC (oracle/tmc_check.c; check d)
 *   k_bg, FFI ................ unbiasedness: same T(r) within errors, E[W] = 1
 *   directional weighting .... Eq. 6-7 (R19): HG normalisation, E[W] = 1, absorbed energy independent of g_S, T(r) of g_E
 *   TMC iteration ............ L29-37 (R22): dies_oracle_tmc_run; pins in tests/test_oracle_tmc.py (independent
 *                              Cartesian TMC, IRE fixed point, closed-form first flight, conservation)
 *   free-path weighting ...... Eq. 8 (R17): closed-form first flight under weighting, absorbed energy per shell
 *                              independent of k_A, k_S, k_A(rho); injected + reweight = escaped + terminated; guard (L119)
 * Parity unpinned: absolute T(r) of the optically thick configs 2 and 3 beyond IRE<->TMC agreement
 * and conservation (no closed form exists).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846

/* ------------------------------------------------------------------ Philox4x32-10
 * Salmon, Moraes, Dror & Shaw 2011 ("Parallel random numbers: as easy as 1, 2, 3"): 10 rounds,
 * multipliers 0xD2511F53 / 0xCD9E8D57, Weyl key increments 0x9E3779B9 / 0xBB67AE85. */
void dies_oracle_philox4x32_10(const uint32_t key_in[2], const uint32_t ctr_in[4], uint32_t out[4])
{
    uint32_t k0 = key_in[0], k1 = key_in[1];
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    for (int round = 0; round < 10; round++) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
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

/* Reading R1: uniform strictly inside (0,1) and exactly representable in fp32 and fp64:
 * (x >> 9) + 0.5 has 24 significant bits.  (The paper's closed interval 0 <= u <= 1, PAPER.md:L55,
 * would allow -ln 0.)  Range [2^-24, 1 - 2^-24]. */
static double uniform_from_word(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* ------------------------------------------------------------------ model */
typedef struct {
    int N, K, nT;
    double *rb, *rho, *mass;           /* N+1, N, N */
    double *kA, *kS, *g;               /* K */
    double *Tg, *eps;                  /* nT */
    double *F;                         /* nT x K row CDFs of the re-emission spectra */
    double *G;                         /* nT x K row CDFs of the emission spectra themselves (TMC dust packages) */
    int has_ext, has_point;
    double *cdf_ext, *cdf_point;       /* K */
    double L_ext, L_point;
    int *fixed_row;                    /* N, rows used in fixed-temperature mode */
} oracle_model;

void dies_oracle_free(oracle_model* o)
{
    if (!o) return;
    free(o->rb); free(o->rho); free(o->mass); free(o->kA); free(o->kS); free(o->g);
    free(o->Tg); free(o->eps); free(o->F); free(o->G); free(o->cdf_ext); free(o->cdf_point); free(o->fixed_row);
    free(o);
}

static double* dup_array(const double* src, size_t n)
{
    double* p = (double*)malloc(n * sizeof(double));
    memcpy(p, src, n * sizeof(double));
    return p;
}

/* Tables ("precalculated lookup tables"; reading R4):
 *   eps_t   = sum_k emis[t][k]                     power emitted per dust mass at T_t
 *   F[t][k] = sum_{j<=k}(emis[t][j]-emis[t-1][j]) / (eps_t - eps_{t-1}),   emis[-1] = 0, eps_{-1} = 0
 * Row t is the spectrum of "the difference between the emission spectra" (L87) of T_t and T_{t-1}. */
oracle_model* dies_oracle_create(int n_shells, const double* r_bounds, const double* rho,
                                 int n_freq, const double* kappa_abs, const double* kappa_sca, const double* g_hg,
                                 int n_T, const double* T_grid, const double* emis)
{
    if (n_shells < 1 || n_freq < 1 || n_T < 1) return NULL;
    for (int i = 0; i < n_shells; i++) if (!(r_bounds[i + 1] > r_bounds[i]) || rho[i] < 0) return NULL;
    if (r_bounds[0] < 0) return NULL;
    oracle_model* o = (oracle_model*)calloc(1, sizeof(oracle_model));
    o->N = n_shells; o->K = n_freq; o->nT = n_T;
    o->rb = dup_array(r_bounds, n_shells + 1);
    o->rho = dup_array(rho, n_shells);
    o->kA = dup_array(kappa_abs, n_freq);
    o->kS = dup_array(kappa_sca, n_freq);
    o->g = dup_array(g_hg, n_freq);
    o->Tg = dup_array(T_grid, n_T);
    o->mass = (double*)malloc(n_shells * sizeof(double));
    for (int i = 0; i < n_shells; i++) {
        double r0 = r_bounds[i], r1 = r_bounds[i + 1];
        o->mass[i] = rho[i] * (4.0 * PI / 3.0) * (r1 * r1 * r1 - r0 * r0 * r0);
    }
    o->eps = (double*)malloc(n_T * sizeof(double));
    o->F = (double*)malloc((size_t)n_T * n_freq * sizeof(double));
    o->G = (double*)malloc((size_t)n_T * n_freq * sizeof(double));
    for (int t = 0; t < n_T; t++) {
        double s = 0.0;
        for (int k = 0; k < n_freq; k++) s += emis[(size_t)t * n_freq + k];
        o->eps[t] = s;
        {
            /* G[t][k] = sum_{j<=k} emis[t][j] / eps_t: the emission spectrum of T_t as a table u -> bin */
            double c = 0.0;
            for (int k = 0; k < n_freq; k++) { c += emis[(size_t)t * n_freq + k]; o->G[(size_t)t * n_freq + k] = s > 0 ? c / s : 1.0; }
            o->G[(size_t)t * n_freq + n_freq - 1] = 1.0;
        }
        if (t > 0 && !(o->eps[t] > o->eps[t - 1])) { dies_oracle_free(o); return NULL; }
        /* normalise by the sum of the differences themselves (= eps_t - eps_{t-1} up to rounding) */
        double tot = 0.0;
        for (int k = 0; k < n_freq; k++) {
            double prev = (t == 0) ? 0.0 : emis[(size_t)(t - 1) * n_freq + k];
            tot += emis[(size_t)t * n_freq + k] - prev;
        }
        double c = 0.0;
        for (int k = 0; k < n_freq; k++) {
            double prev = (t == 0) ? 0.0 : emis[(size_t)(t - 1) * n_freq + k];
            c += emis[(size_t)t * n_freq + k] - prev;
            o->F[(size_t)t * n_freq + k] = c / tot;
        }
        o->F[(size_t)t * n_freq + n_freq - 1] = 1.0;
    }
    o->fixed_row = (int*)calloc(n_shells, sizeof(int));
    return o;
}

static double* make_cdf(const double* w, int K)
{
    double tot = 0.0;
    for (int k = 0; k < K; k++) tot += w[k];
    double* cdf = (double*)malloc(K * sizeof(double));
    double c = 0.0;
    for (int k = 0; k < K; k++) { c += w[k]; cdf[k] = c / tot; }
    cdf[K - 1] = 1.0;
    return cdf;
}

/* Sources: an isotropic external field and a central point source.
 * L_ext = 4 pi R^2 * pi * sum_k J_k: the inward flux of an isotropic field of mean intensity J is
 * pi J (reading R2b).  The source spectrum table maps a uniform number to a frequency bin (L55). */
int dies_oracle_set_sources(oracle_model* o, const double* ext_bin_intensity, double L_point,
                            const double* point_bin_weights)
{
    free(o->cdf_ext); free(o->cdf_point);
    o->cdf_ext = o->cdf_point = NULL;
    o->has_ext = o->has_point = 0;
    o->L_ext = o->L_point = 0.0;
    if (ext_bin_intensity) {
        double J = 0.0;
        for (int k = 0; k < o->K; k++) J += ext_bin_intensity[k];
        if (J > 0) {
            double R = o->rb[o->N];
            o->L_ext = 4.0 * PI * R * R * PI * J;
            o->cdf_ext = make_cdf(ext_bin_intensity, o->K);
            o->has_ext = 1;
        }
    }
    if (point_bin_weights && L_point > 0) {
        o->L_point = L_point;
        o->cdf_point = make_cdf(point_bin_weights, o->K);
        o->has_point = 1;
    }
    return o->has_ext + o->has_point;
}

/* Row of the re-emission table for a cell at emitted power eps per mass:
 * t(eps) = #{j : eps_j <= eps}, clamped to the last row. */
static int row_of_eps(const oracle_model* o, double eps)
{
    int t = 0;
    while (t < o->nT && o->eps[t] <= eps) t++;
    return t < o->nT ? t : o->nT - 1;
}

/* Fixed-temperature tracking mode: the row of shell i is the row of eps(T_i), i.e.
 * #{j : T_j <= T_i} clamped (eps(T) is monotone so this equals t(eps(T_i))). */
int dies_oracle_set_fixed_temperature(oracle_model* o, const double* T)
{
    for (int i = 0; i < o->N; i++) {
        int t = 0;
        while (t < o->nT && o->Tg[t] <= T[i]) t++;
        o->fixed_row[i] = t < o->nT ? t : o->nT - 1;
    }
    return 0;
}

/* Temperature lookup ("new dust temperature ... obtained using precalculated lookup
 * tables"; reading R6): eps -> T by linear interpolation in (ln eps, ln T); clamps counted. */
int dies_oracle_temperature(const oracle_model* o, const double* absorbed, double* T, int* clamp_lo, int* clamp_hi)
{
    *clamp_lo = *clamp_hi = 0;
    for (int i = 0; i < o->N; i++) {
        if (!(o->mass[i] > 0)) { T[i] = 0.0; continue; }
        double eps = absorbed[i] / o->mass[i];
        if (eps < o->eps[0]) { T[i] = o->Tg[0]; (*clamp_lo)++; continue; }
        if (eps >= o->eps[o->nT - 1]) { T[i] = o->Tg[o->nT - 1]; (*clamp_hi)++; continue; }
        int t = 0;
        while (o->eps[t + 1] <= eps) t++;
        double f = (log(eps) - log(o->eps[t])) / (log(o->eps[t + 1]) - log(o->eps[t]));
        T[i] = exp(log(o->Tg[t]) + f * (log(o->Tg[t + 1]) - log(o->Tg[t])));
    }
    return 0;
}

void dies_oracle_get_tables(const oracle_model* o, double* eps, double* F, double* mass)
{
    if (eps) memcpy(eps, o->eps, o->nT * sizeof(double));
    if (F) memcpy(F, o->F, (size_t)o->nT * o->K * sizeof(double));
    if (mass) memcpy(mass, o->mass, o->N * sizeof(double));
}

/* ------------------------------------------------------------------ geometry
 * State: shell i, radius r, direction cosine mu w.r.t. the outward radius.  One step goes to the
 * next shell boundary along the straight line: the inner one if the package moves inward and its
 * impact parameter b is smaller than the inner radius, else the outer one. */
static void shell_step(const double* rb, int i, double r, double mu, double* b2_out, double* l, int* inward)
{
    double b2 = r * r * (1.0 - mu * mu);
    double ri = rb[i], ro = rb[i + 1];
    if (mu < 0.0 && ri > 0.0 && b2 < ri * ri) {
        *inward = 1;
        *l = -r * mu - sqrt(fmax(ri * ri - b2, 0.0));
    } else {
        *inward = 0;
        *l = -r * mu + sqrt(fmax(ro * ro - b2, 0.0));
    }
    *b2_out = b2;
}

/* Move to the boundary found by shell_step.  Returns 1 when the package left the model.
 * Inner boundary of shell 0 with r_0 > 0 is an empty cavity: jump across its chord (reading R10). */
static int cross_boundary(const double* rb, int N, int* i, double* r, double* mu, double b2, int inward,
                          uint64_t* crossings)
{
    if (inward) {
        double rn = rb[*i];
        double c = sqrt(fmax(1.0 - b2 / (rn * rn), 0.0));
        *r = rn;
        if (*i == 0) { *mu = +c; *crossings += 2; }
        else { *mu = -c; *i -= 1; *crossings += 1; }
        return 0;
    }
    double rn = rb[*i + 1];
    *r = rn;
    *mu = sqrt(fmax(1.0 - b2 / (rn * rn), 0.0));
    *i += 1;
    *crossings += 1;
    return *i == N;
}

/* Walk a straight line through the shells without interactions and list the segments:
 * exposed so that the tests can compare with brute-force line/sphere intersections. */
int dies_oracle_chord_walk(int n_shells, const double* rb, int i, double r, double mu, int max_seg,
                           int* seg_shell, double* seg_len, int* n_seg)
{
    uint64_t crossings = 0;
    int n = 0;
    for (;;) {
        double b2, l; int inward;
        shell_step(rb, i, r, mu, &b2, &l, &inward);
        if (n < max_seg) { seg_shell[n] = i; seg_len[n] = l; }
        n++;
        if (cross_boundary(rb, n_shells, &i, &r, &mu, b2, inward, &crossings)) break;
        if (n > 4 * n_shells + 8) return -1;
    }
    *n_seg = n;
    return (int)crossings;
}

/* ------------------------------------------------------------------ run state */
enum { C_PACKAGES = 0, C_CROSSINGS, C_FFI_CROSSINGS, C_SCATTERINGS, C_ABSORPTIONS, C_ESCAPED,
       C_UNINTERACTED, C_TERMINATED, C_EXTRA_BLOCKS, C_CLAMP_HI_SAMPLES, C_N };
enum { D_INJECTED = 0, D_ESCAPED, D_UNINTERACTED, D_TERMINATED, D_REWEIGHT, D_N };
enum { EV_LAUNCH = 0, EV_SCATTER = 1, EV_ABSORB = 2, EV_ESCAPE = 3, EV_TERMINATE = 4, EV_UNINTERACTED = 5 };

typedef struct {
    double* absorbed;      /* N   energy per time absorbed in each shell */
    double* escaped;       /* K   energy per time leaving the model per bin */
    double* reemit;        /* N x K or NULL: re-emitted energy per shell and bin */
    double* pathlen;       /* N or NULL: sum of W * l per shell */
    uint64_t* counters;    /* C_N */
    double* sums;          /* D_N */
} tallies;

typedef struct {
    int32_t* ev; int max_ev; int n_ev;   /* quadruples (type, shell, bin, crossings so far) */
    double margin;                       /* smallest relative distance of any decision from its threshold */
} recorder;

static void rec_event(recorder* rec, int type, int shell, int bin, uint64_t crossings)
{
    if (!rec) return;
    if (rec->n_ev < rec->max_ev) {
        int32_t* e = rec->ev + 4 * rec->n_ev;
        e[0] = type; e[1] = shell; e[2] = bin; e[3] = (int32_t)crossings;
    }
    rec->n_ev++;
}

static void rec_margin(recorder* rec, double a, double b)
{
    if (!rec) return;
    double d = fabs(a - b), m = fmax(fabs(a), fabs(b));
    double rel = m > 0 ? d / m : 0.0;
    if (rel < rec->margin) rec->margin = rel;
}

typedef struct { uint32_t key[2]; uint32_t ctr[4]; } stream;

static void draw_block(stream* s, double u[4])
{
    uint32_t x[4];
    dies_oracle_philox4x32_10(s->key, s->ctr, x);
    s->ctr[2] += 1;
    for (int j = 0; j < 4; j++) u[j] = uniform_from_word(x[j]);
}

/* smallest k with cdf[k] > u */
static int sample_cdf(const double* cdf, int K, double u, recorder* rec)
{
    int k = 0;
    while (k < K - 1 && !(cdf[k] > u)) k++;
    if (rec) { rec_margin(rec, cdf[k], u); if (k > 0) rec_margin(rec, cdf[k - 1], u); }
    return k;
}

/* Henyey-Greenstein deflection cosine ("scattering functions approximated with
 * Henyey-Greenstein functions"; Eq. 6 is the density); inversion of its CDF; g -> 0 is isotropic. */
double dies_oracle_hg_cos(double g, double u)
{
    if (fabs(g) < 1e-3) return 2.0 * u - 1.0;
    double t = (1.0 - g * g) / (1.0 - g + 2.0 * g * u);
    return (1.0 + g * g - t * t) / (2.0 * g);
}

typedef struct {
    uint64_t n_total;        /* packages per active source (reading R2) */
    uint64_t seed;
    uint32_t model_index;
    double k_bg;             /* Eq. 5; 0.5 = unweighted */
    int ffi;                 /* Eq. 9-12 */
    int mode;                /* 0 = full IRE, 1 = fixed temperature */
    const double* kA_w;      /* N or NULL: free-path weighting factor k_A of each shell (Eq. 8; L130: may depend on density) */
    double kS_w;             /* free-path weighting factor k_S (Eq. 8); 1 = unweighted */
    double g_E;              /* Eq. 6: re-emission directions from a Henyey-Greenstein function; 0 = isotropic (unweighted) */
    double g_S;              /* Eq. 7: scattering directions from HG(g_S) about the radial reference direction */
    int use_gS;              /* Eq. 7 is active (g_S = 0 is NOT the plain method, L207) */
    int reemit_cell;         /* L253: re-emit from a random position of the cell volume instead of the absorption site */
    int fp32_tallies;        /* negative control (L155, L179-181): keep the absorbed energy of a cell in single precision */
} run_opts;

/* Henyey-Greenstein density of a direction cosine, Eq. 6: p(mu) = (1/2)(1-g^2)/(1+g^2-2 g mu)^{3/2} */
double dies_oracle_hg_pdf(double g, double mu)
{
    return 0.5 * (1.0 - g * g) / pow(1.0 + g * g - 2.0 * g * mu, 1.5);
}

/* Density-dependent k_A: linear in the logarithm of the density, k_dilute at the lowest
 * density of the model and k_dense at the highest (3.0 and 1.0 in the paper's test); shells without dust get
 * k_dense (they have no opacity).  k_dilute = 0 means the same k_dense everywhere. */
void dies_oracle_kA_profile(const oracle_model* o, double k_dense, double k_dilute, double* kA_w)
{
    double lo = 0.0, hi = 0.0; int any = 0;
    for (int i = 0; i < o->N; i++) if (o->rho[i] > 0.0) {
        double l = log(o->rho[i]);
        if (!any) { lo = hi = l; any = 1; }
        if (l < lo) lo = l;
        if (l > hi) hi = l;
    }
    for (int i = 0; i < o->N; i++) {
        kA_w[i] = k_dense;
        if (k_dilute > 0.0 && o->rho[i] > 0.0 && hi > lo)
            kA_w[i] = k_dense + (k_dilute - k_dense) * (hi - log(o->rho[i])) / (hi - lo);
    }
}

/* Launch direction of a background package (Eq. 2: mu = sqrt(u) w.r.t. the inward
 * normal; L99-103, Eq. 5: mu = u^k_bg with weight W = 2 k_bg mu^(2-1/k_bg); k_bg = 0.5 is Eq. 2).
 * Exposed for the E[W] = 1 and direction-distribution pins. */
/* L85: direction cosine w.r.t. the radius after a deflection by Theta (cosine ct) with azimuth phi about the old
 * direction, whose cosine w.r.t. the radius was mu: mu' = mu cos Theta + sqrt(1 - mu^2) sin Theta cos phi.
 * (The scattering step of the package loop calls this function; it is exported so that a test can pin it to
 * E[mu' | mu] = g mu and the second moment of the Henyey-Greenstein function.) */
double dies_oracle_scatter_direction(double mu, double ct, double phi)
{
    double st = sqrt(fmax(1.0 - ct * ct, 0.0));
    double sm = sqrt(fmax(1.0 - mu * mu, 0.0));
    double m = mu * ct + sm * st * cos(phi);
    if (m > 1.0) m = 1.0;
    if (m < -1.0) m = -1.0;
    return m;
}

void dies_oracle_launch_direction(double u, double k_bg, double* mu_in, double* W)
{
    if (k_bg == 0.5) { *mu_in = sqrt(u); *W = 1.0; }
    else { *mu_in = pow(u, k_bg); *W = 2.0 * k_bg * pow(*mu_in, 2.0 - 1.0 / k_bg); }
}

/* Follow one package from launch to escape. */
static void follow_package(const oracle_model* o, const run_opts* opt, tallies* ta, uint64_t p, recorder* rec)
{
    const int N = o->N, K = o->K;
    stream s;
    s.key[0] = (uint32_t)opt->seed; s.key[1] = (uint32_t)(opt->seed >> 32);
    s.ctr[0] = (uint32_t)p; s.ctr[1] = (uint32_t)(p >> 32); s.ctr[2] = 0; s.ctr[3] = opt->model_index;

    /* which source: ids [0,n) belong to the first active source, [n,2n) to the second (reading R2) */
    int src_is_point;
    if (o->has_ext && o->has_point) src_is_point = (p / opt->n_total) == 1;
    else src_is_point = o->has_point;
    double e = (src_is_point ? o->L_point : o->L_ext) / (double)opt->n_total;   /* L51: equal energies */

    double u[4];
    draw_block(&s, u);
    /* L55: frequency from the source spectrum table */
    int k = sample_cdf(src_is_point ? o->cdf_point : o->cdf_ext, K, u[0], rec);
    double W = 1.0, r, mu;
    int i;
    if (!src_is_point) {
        /* L57-65, Eq. 2: enter at the surface, mu_in = sqrt(u) w.r.t. the inward normal;
         * L99-103, Eq. 5: mu_in = u^k_bg with weight 2 k_bg mu^(2 - 1/k_bg) */
        double mu_in;
        dies_oracle_launch_direction(u[1], opt->k_bg, &mu_in, &W);
        r = o->rb[N]; i = N - 1; mu = -mu_in;
    } else {
        /* L65: isotropic emission from the centre: every direction is radial (reading R9) */
        r = o->rb[0]; i = 0; mu = 1.0;
    }
    /* Eq. 1 */
    double tauS = -log(u[2]);
    double tauA = -log(u[3]);
    const double W_launch = W;
    uint64_t crossings = 0;
    ta->counters[C_PACKAGES] += 1;
    ta->sums[D_INJECTED] += W * e;
    rec_event(rec, EV_LAUNCH, i, k, 0);

    /* Forced first interaction (Eq. 9-12; reading R11) */
    int forced = 0, forced_scatter = 0;
    double tauE = 0.0;
    if (opt->ffi) {
        double tau0 = 0.0;
        {
            int wi = i; double wr = r, wmu = mu; uint64_t wc = 0;
            const double kE = o->kA[k] + o->kS[k];          /* L149: absorption + scattering */
            for (;;) {
                double b2, l; int inward;
                shell_step(o->rb, wi, wr, wmu, &b2, &l, &inward);
                tau0 += kE * o->rho[wi] * l;
                if (cross_boundary(o->rb, N, &wi, &wr, &wmu, b2, inward, &wc)) break;
            }
            ta->counters[C_FFI_CROSSINGS] += wc;
        }
        double P = -expm1(-tau0);                            /* Eq. 12: W = 1 - e^{-tau0} */
        double W_un = W * exp(-tau0);                        /* the share that crosses without interacting */
        ta->escaped[k] += W_un * e;
        ta->sums[D_ESCAPED] += W_un * e;
        ta->sums[D_UNINTERACTED] += W_un * e;
        if (!(tau0 > 0.0)) {
            ta->counters[C_UNINTERACTED] += 1;
            rec_event(rec, EV_UNINTERACTED, i, k, 0);
            return;
        }
        W = W * P;
        tauE = -log1p(-u[2] * P);                            /* Eq. 10 */
        double omega = o->kS[k] / (o->kA[k] + o->kS[k]);
        forced = 1;
        forced_scatter = u[3] < omega;
        rec_margin(rec, u[3], omega);
    }

    for (;;) {
        double b2, l; int inward;
        shell_step(o->rb, i, r, mu, &b2, &l, &inward);
        if (rec && mu < 0.0 && o->rb[i] > 0.0) rec_margin(rec, b2, o->rb[i] * o->rb[i]);
        const double rho = o->rho[i];
        /* Eq. 4; with free-path weighting (L123-130, Eq. 8; reading R17) the two clocks run k_A and k_S times
         * faster than the true optical depths: p'(tau) = k e^{-k tau} */
        const double kAw = opt->kA_w ? opt->kA_w[i] : 1.0, kSw = opt->kS_w;
        double dtauA = kAw * o->kA[k] * rho * l;
        double dtauS = kSw * o->kS[k] * rho * l;
        int event = 0, absorb = 0;
        double l_e = l;
        if (forced) {
            double dtauE = dtauA + dtauS;
            rec_margin(rec, tauE, dtauE);
            if (tauE >= dtauE) tauE -= dtauE;
            else { event = 1; absorb = !forced_scatter; l_e = l * tauE / dtauE; }
        } else {
            rec_margin(rec, tauA, dtauA);
            rec_margin(rec, tauS, dtauS);
            if (tauA >= dtauA && tauS >= dtauS) { tauA -= dtauA; tauS -= dtauS; }
            else {
                /* L85/L87: whichever free path runs out first along the step (reading R7: tie -> absorption) */
                event = 1;
                absorb = tauA * (kSw * o->kS[k]) <= tauS * (kAw * o->kA[k]);
                rec_margin(rec, tauA * (kSw * o->kS[k]), tauS * (kAw * o->kA[k]));
                l_e = absorb ? l * tauA / dtauA : l * tauS / dtauS;
            }
        }
        if (ta->pathlen) ta->pathlen[i] += W * l_e;
        if (kAw != 1.0 || kSw != 1.0) {
            /* Eq. 8 along the step: the true survival probability over the biased one, e^{-dtau} / e^{-k dtau},
             * for both clocks; the event that ends the step adds the factor 1/k of its own clock */
            const double W_old = W;
            W *= exp(((kAw - 1.0) * o->kA[k] + (kSw - 1.0) * o->kS[k]) * rho * l_e);
            if (event && !forced) W /= absorb ? kAw : kSw;
            ta->sums[D_REWEIGHT] += (W - W_old) * e;
        }
        if (!event) {
            if (cross_boundary(o->rb, N, &i, &r, &mu, b2, inward, &crossings)) {
                /* L87 last sentence: the package leaves the model volume */
                ta->escaped[k] += W * e;
                ta->sums[D_ESCAPED] += W * e;
                ta->counters[C_ESCAPED] += 1;
                ta->counters[C_CROSSINGS] += crossings;
                rec_event(rec, EV_ESCAPE, N - 1, k, crossings);
                return;
            }
            continue;
        }
        /* truncate the step at the event position */
        forced = 0;
        {
            double sp = r * mu + l_e;
            double re = sqrt(b2 + sp * sp);
            mu = re > 0.0 ? sp / re : 1.0;
            if (mu > 1.0) mu = 1.0;
            if (mu < -1.0) mu = -1.0;
            r = re;
        }
        if (!absorb) {
            /* L85: scatter with the dust scattering function, redraw both free paths */
            draw_block(&s, u);
            if (opt->use_gS) {
                /* L112-117, Eq. 7 (garbled as printed; reading R19): the new direction is drawn from HG(g_S) about
                 * the radial reference direction (towards the centre for the external field, away from it for the
                 * central source, L109), with a uniform azimuth about that axis; the weight is the ratio of the
                 * dust's HG density at the true scattering angle to the sampling density */
                const double mup = dies_oracle_hg_cos(opt->g_S, u[0]);
                const double phi = 2.0 * PI * u[1];
                const double mu1 = src_is_point ? mup : -mup;
                double ct = mu * mu1 + sqrt(fmax(1.0 - mu * mu, 0.0)) * sqrt(fmax(1.0 - mu1 * mu1, 0.0)) * cos(phi);
                if (ct > 1.0) ct = 1.0;
                if (ct < -1.0) ct = -1.0;
                const double W_old = W;
                W *= dies_oracle_hg_pdf(o->g[k], ct) / dies_oracle_hg_pdf(opt->g_S, mup);
                ta->sums[D_REWEIGHT] += (W - W_old) * e;
                mu = mu1;
            } else {
            mu = dies_oracle_scatter_direction(mu, dies_oracle_hg_cos(o->g[k], u[0]), 2.0 * PI * u[1]);
            }
            tauS = -log(u[2]);
            tauA = -log(u[3]);
            ta->counters[C_SCATTERINGS] += 1;
            rec_event(rec, EV_SCATTER, i, k, crossings);
        } else {
            /* L87: absorb into the current cell, update its temperature, re-emit the same energy
             * at the same position, isotropically, at a frequency drawn from the difference of
             * the emission spectra at the new and old temperatures */
            double old = ta->absorbed[i];
            double new_ = old + W * e;
            /* L155: "the limited precision of floating point operations" -- the paper's fp32 counters stop growing
             * once an update is below half a unit in the last place of the sum (from ~1e8 packages on, L179) */
            if (opt->fp32_tallies) new_ = (double)(float)((float)old + (float)(W * e));
            ta->absorbed[i] = new_;
            int t;
            if (opt->mode == 1) t = o->fixed_row[i];
            else {
                double eps_old = old / o->mass[i], eps_new = new_ / o->mass[i];
                int t_old = row_of_eps(o, eps_old), t_new = row_of_eps(o, eps_new);
                if (t_old != t_new) {
                    /* reading R4: emission spectrum piecewise linear in eps between table rows:
                     * pick eps* uniformly in [eps_old, eps_new) and use the row of eps* */
                    draw_block(&s, u);
                    ta->counters[C_EXTRA_BLOCKS] += 1;
                    t = row_of_eps(o, eps_old + u[0] * (eps_new - eps_old));
                } else t = t_old;
                if (eps_new >= o->eps[o->nT - 1]) ta->counters[C_CLAMP_HI_SAMPLES] += 1;
            }
            draw_block(&s, u);
            k = sample_cdf(o->F + (size_t)t * K, K, u[0], rec);
            mu = 2.0 * u[1] - 1.0;
            if (opt->g_E != 0.0) {
                /* L105-110, Eq. 6: HG(g_E) instead of isotropic, measured from the direction towards the centre
                 * (external field) or away from it (central source); weight = isotropic density / HG density */
                const double mup = dies_oracle_hg_cos(opt->g_E, u[1]);
                const double W_old = W;
                W *= 0.5 / dies_oracle_hg_pdf(opt->g_E, mup);
                ta->sums[D_REWEIGHT] += (W - W_old) * e;
                mu = src_is_point ? mup : -mup;
            }
            tauS = -log(u[2]);
            tauA = -log(u[3]);
            if (opt->reemit_cell) {
                /* L253 (reading R20): "the position of re-emission was randomised within the cell volume":
                 * radius uniform in volume between the boundaries of shell i, one more block for its uniform */
                double u2[4];
                draw_block(&s, u2);
                const double ri = o->rb[i], ro = o->rb[i + 1];
                r = cbrt(ri * ri * ri + u2[0] * (ro * ro * ro - ri * ri * ri));
                if (r < ri) r = ri;
                if (r > ro) r = ro;
            }
            if (ta->reemit) ta->reemit[(size_t)i * K + k] += W * e;
            ta->counters[C_ABSORPTIONS] += 1;
            rec_event(rec, EV_ABSORB, i, k, crossings);
        }
        /* L119: safeguard against trapped packages (never triggers with k_bg/FFI only: W is constant) */
        if (W < 1e-10 * W_launch) {
            ta->sums[D_TERMINATED] += W * e;
            ta->counters[C_TERMINATED] += 1;
            ta->counters[C_CROSSINGS] += crossings;
            rec_event(rec, EV_TERMINATE, i, k, crossings);
            return;
        }
    }
}

/* Run packages first_id .. first_id+n_run-1 of the id space [0, n_sources*n_total) in the order
 * first_id + (j*id_stride mod n_run), j = 0..n_run-1 (id_stride = 1: ascending; any stride coprime
 * to n_run visits every id once -- used by the order-independence pin). Tallies accumulate. */
int dies_oracle_run(const oracle_model* o, uint64_t n_total, uint64_t first_id, uint64_t n_run, uint64_t id_stride,
                    uint64_t seed, uint32_t model_index, double k_bg, int ffi, int mode,
                    const double* kA_w, double kS_w, double g_E, double g_S, int use_gS, int reemit_cell, int fp32_tallies,
                    double* absorbed, double* escaped, double* reemit, double* pathlen,
                    uint64_t* counters, double* sums)
{
    if (!o || !(o->has_ext || o->has_point) || n_total == 0) return -4;
    if (!(k_bg > 0.0) || !(kS_w > 0.0)) return -1;
    if (kA_w) for (int i = 0; i < o->N; i++) if (!(kA_w[i] > 0.0)) return -1;
    if (ffi && (kA_w || kS_w != 1.0)) return -1;             /* alternatives in the paper (Fig. 7), not combined */
    if (!(fabs(g_E) < 1.0) || !(fabs(g_S) < 1.0)) return -1;
    run_opts opt = { n_total, seed, model_index, k_bg, ffi, mode, kA_w, kS_w, g_E, g_S, use_gS, reemit_cell, fp32_tallies };
    tallies ta = { absorbed, escaped, reemit, pathlen, counters, sums };
    for (uint64_t j = 0; j < n_run; j++) {
        uint64_t p = first_id + (uint64_t)(((unsigned __int128)j * id_stride) % n_run);
        follow_package(o, &opt, &ta, p, NULL);
    }
    return 0;
}

/* Replay one package against the given tallies (not modified) and list its events. */
int dies_oracle_trace(const oracle_model* o, uint64_t n_total, uint64_t package_id, uint64_t seed,
                      uint32_t model_index, double k_bg, int ffi, int mode, const double* kA_w, double kS_w,
                      double g_E, double g_S, int use_gS, int reemit_cell, const double* absorbed_state,
                      int32_t* events, int max_events, int* n_events, double* min_margin)
{
    if (!o || !(o->has_ext || o->has_point) || n_total == 0) return -4;
    if (ffi && (kA_w || kS_w != 1.0)) return -1;
    run_opts opt = { n_total, seed, model_index, k_bg, ffi, mode, kA_w, kS_w, g_E, g_S, use_gS, reemit_cell, 0 };
    double* absorbed = (double*)calloc(o->N, sizeof(double));
    double* escaped = (double*)calloc(o->K, sizeof(double));
    if (absorbed_state) memcpy(absorbed, absorbed_state, o->N * sizeof(double));
    uint64_t counters[C_N] = {0};
    double sums[D_N] = {0};
    tallies ta = { absorbed, escaped, NULL, NULL, counters, sums };
    recorder rec = { events, max_events, 0, 1.0 };
    follow_package(o, &opt, &ta, package_id, &rec);
    *n_events = rec.n_ev;
    *min_margin = rec.margin;
    free(absorbed); free(escaped);
    return 0;
}

/* ------------------------------------------------------------------ traditional Monte Carlo (TMC), one iteration
 * "The calculations can be divided into iterations, where the radiation field is estimated using
 * up-to-date information on the radiation sources, including the emission from the dust with its current estimated
 * temperatures.  When the simulation step has been finished, the knowledge of the radiation field is used to update the
 * dust temperatures in every cell."  L37: "the energy absorption is calculated continuously, with updates made to
 * every cell along the photon path between discrete scattering events".  L251: in TMC re-emission "happens uniformly
 * over the cell".  Reading R22:
 *   - every active source sends n_total packages as in the IRE method (L49-65); the dust sends n_total packages of
 *     energy L_dust / n_total, L_dust = sum_i m_i eps_i, eps_i the power per mass cell i emits in its current state;
 *   - a dust package starts in cell i with probability m_i eps_i / L_dust, at a radius uniform in the volume of the
 *     cell, in an isotropic direction, in a bin drawn from the cell's emission spectrum C(eps_i), the cumulative
 *     spectrum of reading R4 (piecewise linear in eps between the rows of the emission table): with probability
 *     eps_{t-1} / eps_i from the spectrum of row t-1 itself, else from the difference spectrum of row t
 *     (t = #{rows with eps_t <= eps_i});
 *   - along a step of length l the package of weight W leaves W (1 - e^{-kappa_A rho l}) in the cell (the integral of
 *     L37's update over the step) and keeps the rest; scatterings are discrete events at tau_S = -ln u (Eq. 1);
 *   - a package ends when it leaves the model, or below 1e-10 of its launch weight (L119).
 * Philox blocks of a package (RNG contract): source package: block 0 = (bin, direction, tau_S, -) as in the IRE method;
 * dust package: block 0 = (cell, radius, direction cosine, row mix), block 1 = (bin, tau_S, -, -); every scattering:
 * (cos Theta, phi, tau_S, -).  Package ids: the sources first ([0, n_total) ...), then the dust.
 * The caller iterates: eps_i <- absorbed_i / m_i until the temperatures stop changing (L31). */
int dies_oracle_tmc_run(const oracle_model* o, uint64_t n_total, uint64_t seed, uint32_t model_index,
                        const double* eps_cur, double* absorbed, double* escaped, uint64_t* counters, double* sums)
{
    if (!o || !(o->has_ext || o->has_point) || n_total == 0) return -4;
    const int N = o->N, K = o->K, nT = o->nT;
    const int n_src = o->has_ext + o->has_point;
    /* the cells as a source table (L55 applied to the dust) */
    double* cellcdf = (double*)malloc(N * sizeof(double));
    double L_dust = 0.0;
    for (int i = 0; i < N; i++) { L_dust += o->mass[i] * (eps_cur ? eps_cur[i] : 0.0); cellcdf[i] = L_dust; }
    if (L_dust > 0.0) { for (int i = 0; i < N; i++) cellcdf[i] /= L_dust; cellcdf[N - 1] = 1.0; }
    const uint64_t n_ids = (uint64_t)(n_src + (L_dust > 0.0 ? 1 : 0)) * n_total;
    for (uint64_t p = 0; p < n_ids; p++) {
        stream s;
        s.key[0] = (uint32_t)seed; s.key[1] = (uint32_t)(seed >> 32);
        s.ctr[0] = (uint32_t)p; s.ctr[1] = (uint32_t)(p >> 32); s.ctr[2] = 0; s.ctr[3] = model_index;
        const int which = (int)(p / n_total);                 /* 0 .. n_src-1: sources; n_src: dust */
        double u[4], e, r, mu, tauS;
        int i, k;
        draw_block(&s, u);
        if (which < n_src) {
            const int src_is_point = (o->has_ext && o->has_point) ? which == 1 : o->has_point;
            e = (src_is_point ? o->L_point : o->L_ext) / (double)n_total;
            k = sample_cdf(src_is_point ? o->cdf_point : o->cdf_ext, K, u[0], NULL);
            if (!src_is_point) { r = o->rb[N]; i = N - 1; mu = -sqrt(u[1]); }            /* Eq. 2 */
            else { r = o->rb[0]; i = 0; mu = 1.0; }                                      /* L65, R9 */
            tauS = -log(u[2]);
        } else {
            e = L_dust / (double)n_total;
            i = sample_cdf(cellcdf, N, u[0], NULL);
            const double ri = o->rb[i], ro = o->rb[i + 1];
            r = cbrt(ri * ri * ri + u[1] * (ro * ro * ro - ri * ri * ri));               /* L251: uniform over the cell */
            if (r < ri) r = ri;
            if (r > ro) r = ro;
            mu = 2.0 * u[2] - 1.0;
            const double eps = eps_cur[i];
            int t = 0;
            while (t < nT && o->eps[t] <= eps) t++;                                      /* #{rows with eps_t <= eps} */
            const double* cdf;
            if (t >= nT) cdf = o->G + (size_t)(nT - 1) * K;                              /* beyond the table: its last row */
            else if (t > 0 && u[3] < o->eps[t - 1] / eps) cdf = o->G + (size_t)(t - 1) * K;
            else cdf = o->F + (size_t)t * K;
            double v[4];
            draw_block(&s, v);
            k = sample_cdf(cdf, K, v[0], NULL);
            tauS = -log(v[1]);
        }
        double W = 1.0;
        uint64_t crossings = 0;
        counters[C_PACKAGES] += 1;
        sums[D_INJECTED] += e;
        for (;;) {
            double b2, l; int inward;
            shell_step(o->rb, i, r, mu, &b2, &l, &inward);
            const double rho = o->rho[i];
            const double dtauS = o->kS[k] * rho * l;
            const int event = !(tauS >= dtauS);
            const double l_e = event ? l * tauS / dtauS : l;
            /* L37: continuous absorption along the step */
            const double dep = W * -expm1(-o->kA[k] * rho * l_e);
            absorbed[i] += e * dep;
            W -= dep;
            if (!event) {
                tauS -= dtauS;
                if (cross_boundary(o->rb, N, &i, &r, &mu, b2, inward, &crossings)) {
                    escaped[k] += W * e;
                    sums[D_ESCAPED] += W * e;
                    counters[C_ESCAPED] += 1;
                    break;
                }
            } else {
                double sp = r * mu + l_e;
                double re = sqrt(b2 + sp * sp);
                mu = re > 0.0 ? sp / re : 1.0;
                if (mu > 1.0) mu = 1.0;
                if (mu < -1.0) mu = -1.0;
                r = re;
                draw_block(&s, u);
                mu = dies_oracle_scatter_direction(mu, dies_oracle_hg_cos(o->g[k], u[0]), 2.0 * PI * u[1]);
                tauS = -log(u[2]);
                counters[C_SCATTERINGS] += 1;
            }
            if (W < 1e-10) {                                   /* L119 */
                sums[D_TERMINATED] += W * e;
                counters[C_TERMINATED] += 1;
                break;
            }
        }
        counters[C_CROSSINGS] += crossings;
    }
    free(cellcdf);
    return 0;
}


double dies_oracle_uniform(uint32_t x) { return uniform_from_word(x); }
