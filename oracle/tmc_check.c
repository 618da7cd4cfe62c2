/*
 * tmc_check.c -- TEST INFRASTRUCTURE: pin (d) of the oracle ("agreement with a traditional
 * Monte Carlo iteration to convergence on config 1", BASELINE.json north_star).
 *
 * A minimal traditional Monte Carlo (TMC): per iteration the external field
 * and the dust emission at the current temperatures are simulated with packages of fixed frequency,
 * absorption is accumulated CONTINUOUSLY along the paths (L37 "updates made to every cell along the
 * photon path between discrete scattering events"), scatterings are discrete events, and the
 * temperatures are updated at the end of the iteration; repeat to convergence (L31).
 *
 * Deliberately independent of dies_oracle.c: geometry is 3-D Cartesian (position and direction
 * vectors, line/sphere quadratics), the random numbers come from splitmix64/xoshiro256**, and
 * nothing is shared with or included from the oracle or the CUDA path.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define PI 3.14159265358979323846

typedef struct { uint64_t s[4]; } rng_t;
static uint64_t splitmix(uint64_t* x) { uint64_t z = (*x += 0x9E3779B97F4A7C15ull); z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; return z ^ (z >> 31); }
static uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static uint64_t next(rng_t* r) { uint64_t* s = r->s; uint64_t res = rotl(s[1] * 5, 7) * 9, t = s[1] << 17; s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45); return res; }
static double uni(rng_t* r) { return ((double)(next(r) >> 11) + 0.5) * (1.0 / 9007199254740992.0); }

/* distance along the ray x + t d to the sphere of radius R: smallest t > tmin, or -1 */
static double hit(const double x[3], const double d[3], double R, double tmin)
{
    double xd = x[0] * d[0] + x[1] * d[1] + x[2] * d[2];
    double xx = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
    double disc = xd * xd - (xx - R * R);
    if (disc < 0) return -1.0;
    double sq = sqrt(disc);
    double t1 = -xd - sq, t2 = -xd + sq;
    if (t1 > tmin) return t1;
    if (t2 > tmin) return t2;
    return -1.0;
}

static void scatter_dir(double d[3], double ct, double phi)
{
    double st = sqrt(fmax(0.0, 1.0 - ct * ct)), cp = cos(phi), sp = sin(phi);
    double n[3];
    if (fabs(d[2]) > 0.99999) {
        n[0] = st * cp; n[1] = st * sp; n[2] = d[2] > 0 ? ct : -ct;
    } else {
        double q = sqrt(1.0 - d[2] * d[2]);
        n[0] = st * (d[0] * d[2] * cp - d[1] * sp) / q + d[0] * ct;
        n[1] = st * (d[1] * d[2] * cp + d[0] * sp) / q + d[1] * ct;
        n[2] = -st * cp * q + d[2] * ct;
    }
    double nn = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    d[0] = n[0] / nn; d[1] = n[1] / nn; d[2] = n[2] / nn;
}

static int pick(const double* w, int K, double tot, double u)
{
    double c = 0.0, target = u * tot;
    for (int k = 0; k < K; k++) { c += w[k]; if (c > target) return k; }
    return K - 1;
}

/* follow one package of weight (energy/time) E0 in bin k; add absorbed energy to A[] */
static void follow(rng_t* rg, int N, const double* rb, const double* rho, double kA, double kS, double g,
                   double x[3], double d[3], int i, double E0, double* A)
{
    double w = E0;
    double tauS = -log(uni(rg));
    for (int guard = 0; guard < 100000000; guard++) {
        /* next boundary of shell i: inner sphere (if any) or outer sphere */
        double tin = rb[i] > 0 ? hit(x, d, rb[i], 1e-14 * rb[N]) : -1.0;
        double tout = hit(x, d, rb[i + 1], 1e-14 * rb[N]);
        int inward = 0; double t = tout;
        /* the inner sphere is hit first only if we move inward */
        double xd = x[0] * d[0] + x[1] * d[1] + x[2] * d[2];
        if (tin > 0 && xd < 0 && tin < tout) { t = tin; inward = 1; }
        if (t < 0) t = 0;
        double dS = kS * rho[i] * t;
        int scat = 0;
        if (dS > tauS) { t *= tauS / dS; scat = 1; }
        double dA = kA * rho[i] * t;
        double absorbed = w * (-expm1(-dA));
        A[i] += absorbed;
        w -= absorbed;
        for (int c = 0; c < 3; c++) x[c] += t * d[c];
        if (scat) {
            double u = uni(rg), ct;
            if (fabs(g) < 1e-3) ct = 2 * u - 1;
            else { double q = (1 - g * g) / (1 - g + 2 * g * u); ct = (1 + g * g - q * q) / (2 * g); }
            scatter_dir(d, ct, 2 * PI * uni(rg));
            tauS = -log(uni(rg));
            continue;
        }
        tauS -= dS;
        if (inward) {
            if (i == 0) {   /* empty cavity: fly across */
                double tc = hit(x, d, rb[0], 1e-14 * rb[N]);
                if (tc > 0) for (int c = 0; c < 3; c++) x[c] += tc * d[c];
            } else i -= 1;
        } else {
            i += 1;
            if (i == N) return;
        }
        if (w < 1e-30 * E0) return;
    }
}

static double T_of_eps(int nT, const double* Tg, const double* eps, double e)
{
    if (e <= eps[0]) return Tg[0];
    if (e >= eps[nT - 1]) return Tg[nT - 1];
    int t = 0;
    while (eps[t + 1] <= e) t++;
    double f = (log(e) - log(eps[t])) / (log(eps[t + 1]) - log(eps[t]));
    return exp(log(Tg[t]) + f * (log(Tg[t + 1]) - log(Tg[t])));
}

/* Returns the number of iterations used.  T_out: N converged temperatures. */
int tmc_solve(int N, const double* rb, const double* rho, int K, const double* kA, const double* kS, const double* g,
              int nT, const double* Tg, const double* emis, const double* ext_bin_intensity,
              uint64_t n_src, uint64_t n_dust, int max_iter, double tol, uint64_t seed, double* T_out)
{
    rng_t rg; uint64_t sm = seed;
    for (int j = 0; j < 4; j++) rg.s[j] = splitmix(&sm);
    double* eps = (double*)calloc(nT, sizeof(double));
    for (int t = 0; t < nT; t++) for (int k = 0; k < K; k++) eps[t] += emis[(size_t)t * K + k];
    double* mass = (double*)calloc(N, sizeof(double));
    for (int i = 0; i < N; i++) mass[i] = rho[i] * 4.0 * PI / 3.0 * (pow(rb[i + 1], 3) - pow(rb[i], 3));
    double* A_src = (double*)calloc(N, sizeof(double));
    double* A = (double*)calloc(N, sizeof(double));
    double* ecell = (double*)calloc(N, sizeof(double));
    double* spec = (double*)calloc(K, sizeof(double));
    const double R = rb[N];
    double Jtot = 0.0;
    for (int k = 0; k < K; k++) Jtot += ext_bin_intensity[k];
    const double L = 4.0 * PI * R * R * PI * Jtot;

    /* external field: simulated once (it does not depend on the temperatures) */
    for (uint64_t p = 0; p < n_src; p++) {
        int k = pick(ext_bin_intensity, K, Jtot, uni(&rg));
        double mu = sqrt(uni(&rg)), phi = 2 * PI * uni(&rg), st = sqrt(1 - mu * mu);
        double x[3] = { 0, 0, -R * (1.0 - 1e-13) }, d[3] = { cos(phi) * st, sin(phi) * st, mu };
        follow(&rg, N, rb, rho, kA[k], kS[k], g[k], x, d, N - 1, L / (double)n_src, A_src);
    }
    for (int i = 0; i < N; i++) { ecell[i] = mass[i] > 0 ? A_src[i] / mass[i] : 0; T_out[i] = T_of_eps(nT, Tg, eps, ecell[i]); }

    int it;
    for (it = 1; it <= max_iter; it++) {
        for (int i = 0; i < N; i++) A[i] = A_src[i];
        /* dust emission: same number of packages from every cell, weight = cell luminosity / count */
        uint64_t per_cell = n_dust / N > 0 ? n_dust / N : 1;
        for (int i = 0; i < N; i++) {
            double e = ecell[i];
            if (!(mass[i] > 0) || !(e > 0)) continue;
            /* emission spectrum at eps = e: rows interpolated linearly in eps */
            double tot = 0;
            if (e <= eps[0]) { for (int k = 0; k < K; k++) { spec[k] = emis[k] * e / eps[0]; tot += spec[k]; } }
            else {
                int t = 0;
                while (t + 1 < nT - 1 && eps[t + 1] <= e) t++;
                double f = (e - eps[t]) / (eps[t + 1] - eps[t]);
                if (f > 1) f = 1;
                for (int k = 0; k < K; k++) { spec[k] = emis[(size_t)t * K + k] + f * (emis[(size_t)(t + 1) * K + k] - emis[(size_t)t * K + k]); tot += spec[k]; }
            }
            double Lcell = mass[i] * e;
            for (uint64_t p = 0; p < per_cell; p++) {
                int k = pick(spec, K, tot, uni(&rg));
                double r3 = pow(rb[i], 3) + uni(&rg) * (pow(rb[i + 1], 3) - pow(rb[i], 3));
                double r = cbrt(r3);
                if (r >= rb[i + 1]) r = rb[i + 1] * (1 - 1e-13);
                if (r <= rb[i]) r = rb[i] + 1e-13 * rb[N];
                double cz = 2 * uni(&rg) - 1, ph = 2 * PI * uni(&rg), sz = sqrt(1 - cz * cz);
                double x[3] = { 0, 0, r }, d[3] = { sz * cos(ph), sz * sin(ph), cz };
                follow(&rg, N, rb, rho, kA[k], kS[k], g[k], x, d, i, Lcell / (double)per_cell, A);
            }
        }
        double worst = 0;
        for (int i = 0; i < N; i++) {
            double e = mass[i] > 0 ? A[i] / mass[i] : 0;
            double Tn = T_of_eps(nT, Tg, eps, e);
            double rel = fabs(Tn - T_out[i]) / Tn;
            if (rel > worst) worst = rel;
            ecell[i] = e; T_out[i] = Tn;
        }
        if (worst < tol) break;
    }
    free(eps); free(mass); free(A_src); free(A); free(ecell); free(spec);
    return it;
}
