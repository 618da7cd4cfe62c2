// dies_lib.cu -- C ABI of libdies (include/dies.h): host argument checking, device table construction,
// launches of the trackers (dies_fly.cuh: runs with weights fixed at launch; dies_tracker.cuh: runs with free-path or
// directional weighting) and read-back.  Compiled for sm_100a only; no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/dies.h"
#include "dies_tracker.cuh"
#include "dies_fly.cuh"
#include "dies_tmc.cuh"

using namespace dies;

// ------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
#define CUDA_TRY(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess) return fail(DIES_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
    } while (0)

extern "C" const char* dies_last_error(void) { return g_err; }

// ------------------------------------------------------------------ workspace layout
struct Layout {
    size_t G, epscur, cellcdf, tmcrow, tmcmix, Ldust, qsdust;      // TMC mode (dies_tmc.cuh)
    size_t emis, eps, Tgrid, epsgrid, F, guideF, guideS, stabW, bintab, omega, dustin, rb, rho, mass, stab, cscale, srccdf, srcin, Lsrc, mp,
        fixed_row, Tfix, A, esc, next_id, counters, ticket, T_out, Lesc_out, eunit, flags, epsref, total;
};
static size_t al(size_t x) { return (x + 255) & ~(size_t)255; }
static Layout make_layout(int N, int K, int nT, int M)
{
    Layout L;
    const size_t ldS = (size_t)N + 1;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = al(o + bytes); return at; };
    L.emis = take((size_t)nT * K * 8);
    L.eps = take((size_t)nT * 8);
    L.Tgrid = take((size_t)nT * 8);
    L.epsgrid = take((size_t)nT * 4);
    L.F = take((size_t)nT * K * 4);
    L.G = take((size_t)nT * K * 4);
    L.epscur = take((size_t)M * ldS * 8);
    L.cellcdf = take((size_t)M * ldS * 4);
    L.tmcrow = take((size_t)M * ldS * 4);
    L.tmcmix = take((size_t)M * ldS * 4);
    L.Ldust = take((size_t)M * 8);
    L.qsdust = take((size_t)M * 4);
    L.guideF = take((size_t)nT * kGuide * 2);
    L.guideS = take((size_t)M * 2 * kGuide * 2);
    L.stabW = take((size_t)M * 2 * (ldS + 1) * 16);
    L.bintab = take((size_t)K * 16);
    L.omega = take((size_t)K * 4);
    L.dustin = take((size_t)3 * K * 8);
    L.rb = take((size_t)M * (N + 1) * 8);
    L.rho = take((size_t)M * N * 8);
    L.mass = take((size_t)M * ldS * 8);
    L.stab = take((size_t)M * 2 * (ldS + 1) * 8);
    L.cscale = take((size_t)M * ldS * 8);
    L.srccdf = take((size_t)M * 2 * K * 4);
    L.srcin = take((size_t)M * 2 * K * 8);
    L.Lsrc = take((size_t)M * 2 * 8);
    L.mp = take((size_t)M * sizeof(ModelParams));
    L.fixed_row = take((size_t)M * ldS * 4);
    L.Tfix = take((size_t)M * N * 8);
    L.A = take((size_t)M * ldS * kTallyStride * 8);
    L.esc = take((size_t)M * K * 8);
    L.next_id = take((size_t)M * 8);
    L.counters = take((size_t)DIES_N_COUNTERS * 8);
    L.ticket = take(16);
    L.T_out = take((size_t)M * N * 8);
    L.Lesc_out = take((size_t)M * K * 8);
    L.eunit = take((size_t)M * 8);
    L.flags = take(64);
    L.epsref = take(16);
    L.total = o;
    return L;
}

struct dies_model {
    int N, K, nT, M, ldS;
    Layout L;
    unsigned char* ws;
    DeviceModel D;
    bool sources_set, fixed_set, ran;
    bool finalized;                       // T_out / Lesc_out / derived counters are those of the last run
    std::vector<double> L_point;          // per model
    std::vector<int> has_ext, has_point;
    unsigned long long done, n_total;     // packages per source already followed / planned
    unsigned long long next_first;        // dies_seek: first package id (per source) of the next fresh run
    int shift;
    int last_mode;                        // mode of the last run (its tallies are in that mode's energy unit)
    uint32_t model0;                      // dies_set_model_offset
    int visit_auto;                       // crossing blocks per crossing phase, from the counters of the last read-out
    cudaStream_t stream;
    int grid_max, blocks_per_sm, n_sms;
    int pool;                             // pool slots per warp of the tracker
    double kref;                          // opacity unit of the device tables: max_k(kappa_abs + kappa_sca)
    size_t smem_bytes, smem_trace_bytes;
    unsigned long long launches;
};

template <class T>
static T* wsp(dies_model* m, size_t off) { return reinterpret_cast<T*>(m->ws + off); }

// ------------------------------------------------------------------ table construction kernels
// eps_t = sum_k emis[t][k];  F[t][k] = cumsum_k(emis[t] - emis[t-1]) / sum_k(emis[t] - emis[t-1])   (R4)
__global__ void k_build_tables(const double* __restrict__ emis, int nT, int K, double* __restrict__ eps,
                               float* __restrict__ F, float* __restrict__ G, int* flags)
{
    // one warp per temperature row: lane l owns the bins [l c, (l+1) c), c = ceil(K / 32)
    const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (t >= nT) return;
    const double* row = emis + (size_t)t * K;
    const double* prev = t > 0 ? row - K : nullptr;
    const int c = (K + 31) / 32, k0 = min(lane * c, K), k1 = min(k0 + c, K);
    double s = 0.0, part = 0.0;
    bool bad = false;
    for (int k = k0; k < k1; k++) {
        const double d = row[k] - (prev ? prev[k] : 0.0);
        if (!(d >= 0.0)) bad = true;
        s += row[k];
        part += d;
    }
    // totals and the exclusive prefix of the partial sums of the increments
    double tot = part, ssum = s, pre = part, pres = s;
    for (int o = 1; o < 32; o <<= 1) {
        const double v = __shfl_up_sync(0xffffffffu, pre, o), vs = __shfl_up_sync(0xffffffffu, pres, o);
        if (lane >= o) { pre += v; pres += vs; }
    }
    pres -= s;
    for (int o = 16; o > 0; o >>= 1) { tot += __shfl_xor_sync(0xffffffffu, tot, o); ssum += __shfl_xor_sync(0xffffffffu, ssum, o); }
    pre -= part;
    if (__any_sync(0xffffffffu, bad) || !(tot > 0.0)) { if (lane == 0) atomicOr(flags, 1); }
    if (lane == 0) eps[t] = ssum;
    float* f = F + (size_t)t * K;
    float* gt = G + (size_t)t * K;                           // the spectrum of T_t itself (TMC dust packages, R22)
    double cum = pre, cums = pres;
    for (int k = k0; k < k1; k++) {
        cum += row[k] - (prev ? prev[k] : 0.0);
        cums += row[k];
        f[k] = (k == K - 1) ? 1.0f : (float)(cum / tot);
        gt[k] = (k == K - 1 || !(ssum > 0.0)) ? 1.0f : (float)(cums / ssum);
    }
}

// guide tables of the cut-point sampler: guide[row][c] = smallest k with cdf[row][k] > c / kGuide
__global__ void k_build_guide(const float* __restrict__ cdf, int n_rows, int K, unsigned short* __restrict__ guide)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_rows * kGuide) return;
    const int row = idx / kGuide, c = idx % kGuide;
    const float u = (float)c / (float)kGuide;
    const float* f = cdf + (size_t)row * K;
    int lo = 0, hi = K - 1;               // cdf[K-1] = 1 > u
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (f[mid] > u) hi = mid; else lo = mid + 1; }
    guide[idx] = (unsigned short)lo;
}

__global__ void k_build_epsgrid(const double* __restrict__ eps, int nT, float* __restrict__ grid, double* epsref,
                                int* flags)
{
    const double ref = sqrt(eps[0] * eps[nT - 1]);
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t == 0) *epsref = ref;
    if (t >= nT) return;
    if (t > 0 && !(eps[t] > eps[t - 1])) atomicOr(flags, 2);
    grid[t] = (float)(eps[t] / ref);
}

// dust table: opacities in units of kappa_ref = max_k(kappa_abs + kappa_sca)
__global__ void k_build_dust(const double* __restrict__ dustin, int K, double kref, float4* bintab, float* omega)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const double ka = dustin[k] / kref, ks = dustin[K + k] / kref, g = dustin[2 * K + k];
    bintab[k] = make_float4((float)(1.0 / ka), (float)(1.0 / ks), (float)g, (float)(ka + ks));   // 1/0 = inf: never hit
    omega[k] = (ka + ks) > 0 ? (float)(ks / (ka + ks)) : 0.f;
}

// shells: lengths in units of the outer radius R, densities as rho^ = rho R kappa_ref; internal shell 0 is the
// empty cavity when r_bounds[0] > 0 (R10).  The table is unfolded along a chord (see DeviceModel in
// dies_tracker.cuh): entry c in [-ldS, ldS+1] = {(r_|c|/R)^2, rho^ of the shell traversed on the way to that
// surface, sign bit = inward}; entry Np+1 is the sentinel {-1, +0}.
__global__ void k_build_shells(const double* __restrict__ rb, const double* __restrict__ rho, int N, int M, double kref,
                               float2* stab, double* mass, ModelParams* mp)
{
    const int ldS = N + 1, ldT = 2 * ldS + 2;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= M * ldT) return;
    const int m = idx / ldT, x = idx % ldT;
    const double* r = rb + (size_t)m * (N + 1);
    const double* d = rho + (size_t)m * N;
    const double R = r[N];
    const int cav = r[0] > 0.0 ? 1 : 0;
    const int Np = N + cav;
    // internal boundary b in [0, Np]: radius 0 at the centre, then the user's boundaries
    auto radius = [&](int b) { return b == 0 ? 0.0 : r[b - cav]; };
    // internal shell j in [0, Np): the cavity (if any) has no dust
    auto dens = [&](int j) { const int i = j - cav; return (i < 0 || i >= N) ? 0.0 : d[i]; };
    if (x == 0) {
        ModelParams p = mp[m];
        p.Np = Np; p.cav = cav; p.r0hat = (float)(r[0] / R);
        double colsum = 0.0;                                              // radial column centre -> surface
        for (int j = 0; j < Np; j++) colsum += dens(j) * kref * (radius(j + 1) - radius(j));
        p.colmax = (float)(2.5 * colsum + 1e-30);                         // > column of the diameter (2 colsum)
        mp[m] = p;
    }
    const int c = x - ldS, a = c < 0 ? -c : c;
    float2 e = make_float2(4.0f, 0.0f);                                  // never read
    if (c <= 0 && a <= Np) {
        const double rr = radius(a) / R;
        const float dh = (float)(dens(a) * R * kref);
        e = make_float2((float)(rr * rr), __int_as_float(__float_as_int(dh) | 0x80000000));
    } else if (c > 0 && c <= Np) {
        const double rr = radius(c) / R;
        e = make_float2((float)(rr * rr), (float)(dens(c - 1) * R * kref));
    } else if (c == Np + 1) {
        e = make_float2(-1.0f, 0.0f);                                    // sentinel: d = -1 - b^2 < 0 stops the package
    }
    stab[(size_t)m * ldT + x] = e;
    if (x < ldS) {
        const int j = x;
        const double pi = 3.14159265358979323846;
        double ms = 0.0;
        if (j < Np) {
            const double r_in = radius(j), r_out = radius(j + 1);
            ms = dens(j) * (4.0 * pi / 3.0) * (r_out * r_out * r_out - r_in * r_in * r_in);
        }
        mass[(size_t)m * ldS + j] = ms;
    }
}

// Shell table of a run with free-path weighting (Eq. 8; R17): the same unfolded table with 16-byte entries
// {(r/R)^2, +-rho^, k_A,i rho^, k_A,i}.  k_A,i is k_dense everywhere, or linear in log(rho) between k_dense at the
// highest density of the model and k_dilute at the lowest (k_dilute > 0).
__global__ void k_build_wshells(const double* __restrict__ rb, const double* __restrict__ rho, int N, int M, double kref,
                                double k_dense, double k_dilute, float4* stabW)
{
    const int ldS = N + 1, ldT = 2 * ldS + 2;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= M * ldT) return;
    const int m = idx / ldT, x = idx % ldT;
    const double* r = rb + (size_t)m * (N + 1);
    const double* d = rho + (size_t)m * N;
    const double R = r[N];
    const int cav = r[0] > 0.0 ? 1 : 0;
    const int Np = N + cav;
    double lo = 0.0, hi = 0.0; bool any = false;
    for (int i = 0; i < N; i++) if (d[i] > 0.0) {
        const double l = log(d[i]);
        if (!any) { lo = hi = l; any = true; }
        lo = fmin(lo, l); hi = fmax(hi, l);
    }
    auto radius = [&](int b) { return b == 0 ? 0.0 : r[b - cav]; };
    auto dens = [&](int j) { const int i = j - cav; return (i < 0 || i >= N) ? 0.0 : d[i]; };
    auto kA = [&](int j) {
        const double dj = dens(j);
        if (k_dilute > 0.0 && dj > 0.0 && hi > lo) return k_dense + (k_dilute - k_dense) * (hi - log(dj)) / (hi - lo);
        return k_dense;
    };
    const int c = x - ldS, a = c < 0 ? -c : c;
    float4 e = make_float4(4.0f, 0.0f, 0.0f, 1.0f);                     // never read
    if (c <= 0 && a <= Np) {
        const double rr = radius(a) / R;
        const float dh = (float)(dens(a) * R * kref);
        e = make_float4((float)(rr * rr), __int_as_float(__float_as_int(dh) | 0x80000000),
                        (float)(kA(a) * dens(a) * R * kref), (float)kA(a));
    } else if (c > 0 && c <= Np) {
        const double rr = radius(c) / R;
        e = make_float4((float)(rr * rr), (float)(dens(c - 1) * R * kref), (float)(kA(c - 1) * dens(c - 1) * R * kref),
                        (float)kA(c - 1));
    } else if (c == Np + 1) {
        e = make_float4(-1.0f, 0.0f, 0.0f, 1.0f);                        // sentinel
    }
    stabW[(size_t)m * ldT + x] = e;
}

// source spectrum tables and luminosities: L_ext = 4 pi R^2 * pi * sum_k J_k
__global__ void k_build_sources(const double* __restrict__ srcin, const double* __restrict__ rb, int N, int K, int M,
                                float* srccdf, double* Lsrc, ModelParams* mp)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * M) return;
    const int m = idx >> 1, which = idx & 1;
    const double* w = srcin + ((size_t)m * 2 + which) * K;
    float* cdf = srccdf + ((size_t)m * 2 + which) * K;
    double tot = 0.0;
    for (int k = 0; k < K; k++) tot += w[k];
    if (which == 0) {
        const double pi = 3.14159265358979323846;
        const double R = rb[(size_t)m * (N + 1) + N];
        Lsrc[2 * m] = 4.0 * pi * R * R * pi * tot;
        mp[m].has_ext = tot > 0.0 ? 1 : 0;                       // which sources of the model are active (R2)
    } else {
        mp[m].has_point = (Lsrc[2 * m + 1] > 0.0 && tot > 0.0) ? 1 : 0;
    }
    double c = 0.0;
    for (int k = 0; k < K; k++) {
        c += w[k];
        cdf[k] = tot > 0.0 ? (float)(c / tot) : 1.0f;
    }
    cdf[K - 1] = 1.0f;
}

// The same tables, one block per (model, source): the weights are staged in shared memory by all threads, thread 0 runs
// the two serial sums there (the SAME order of additions as k_build_sources, so the tables are bit-identical), and the
// divisions and the stores are spread over the block.  k_build_sources walks global memory with one thread per source
// and takes 37 us for the 200 bins of config 2, a tenth of a whole end-to-end step of config 1.
__global__ void k_build_sources_staged(const double* __restrict__ srcin, const double* __restrict__ rb, int N, int K, int M,
                                       float* srccdf, double* Lsrc, ModelParams* mp)
{
    extern __shared__ double s_w[];               // K weights, then their running sums in place
    __shared__ double s_tot;
    const int idx = blockIdx.x;
    const int m = idx >> 1, which = idx & 1;
    const double* w = srcin + ((size_t)m * 2 + which) * K;
    float* cdf = srccdf + ((size_t)m * 2 + which) * K;
    for (int k = threadIdx.x; k < K; k += blockDim.x) s_w[k] = w[k];
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < K; k++) tot += s_w[k];
        if (which == 0) {
            const double pi = 3.14159265358979323846;
            const double R = rb[(size_t)m * (N + 1) + N];
            Lsrc[2 * m] = 4.0 * pi * R * R * pi * tot;
            mp[m].has_ext = tot > 0.0 ? 1 : 0;                   // which sources of the model are active (R2)
        } else {
            mp[m].has_point = (Lsrc[2 * m + 1] > 0.0 && tot > 0.0) ? 1 : 0;
        }
        double c = 0.0;
        for (int k = 0; k < K; k++) { c += s_w[k]; s_w[k] = c; }
        s_tot = tot;
    }
    __syncthreads();
    const double tot = s_tot;
    for (int k = threadIdx.x; k < K; k += blockDim.x)
        cdf[k] = (k == K - 1) ? 1.0f : (tot > 0.0 ? (float)(s_w[k] / tot) : 1.0f);
}

// fixed-temperature rows: #{t : T_grid[t] <= T} clamped
__global__ void k_fixed_rows(const double* __restrict__ Tfix, const double* __restrict__ Tgrid, int nT, int N, int M,
                             const ModelParams* mp, int* fixed_row)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= M * N) return;
    const int m = idx / N, i = idx % N;
    const double T = Tfix[idx];
    int lo = 0, hi = nT;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (Tgrid[mid] > T) hi = mid; else lo = mid + 1; }
    fixed_row[(size_t)m * (N + 1) + i + mp[m].cav] = min(lo, nT - 1);
}

// per run: energy scale of the raw tallies, zeroing, counters
// TMC mode (dies_tmc.cuh; R22): the state of the dust for the next iteration from the tallies of the run before:
// eps_i = absorbed_i / m_i (0 before any run), the cells as a source table, the table row and the mixing share of every
// cell's spectrum C(eps_i), the dust luminosity.  One thread per model; runs before k_prepare_run rescales the tallies.
__global__ void k_tmc_prepare(DeviceModel D, const double* __restrict__ mass, const double* __restrict__ eunit,
                              const double* __restrict__ eps, int have_state, double* epscur, float* cellcdf, int* row,
                              float* mix, double* Ldust)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= D.n_models) return;
    const int ldS = D.ldS, nT = D.nT, Np = D.mp[m].Np;
    double L = 0.0;
    for (int j = 0; j < ldS; j++) {
        const size_t x = (size_t)m * ldS + j;
        const double ms = j < Np ? mass[x] : 0.0;
        const double e = (have_state && ms > 0.0) ? (double)D.A[x * kTallyStride] * eunit[m] / ms : 0.0;
        epscur[x] = e;
        int lo = 0, hi = nT;                           // #{rows with eps_t <= e}
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (eps[mid] > e) hi = mid; else lo = mid + 1; }
        row[x] = lo;
        mix[x] = lo == 0 ? 0.f : (lo >= nT ? 1.f : (float)(eps[lo - 1] / e));
        L += ms * e;
    }
    Ldust[m] = L;
    double c = 0.0;
    for (int j = 0; j < ldS; j++) {
        const size_t x = (size_t)m * ldS + j;
        c += (j < Np ? mass[x] : 0.0) * epscur[x];
        cellcdf[x] = L > 0.0 ? (float)(c / L) : 1.f;
    }
    if (L > 0.0) for (int j = Np - 1; j < ldS; j++) cellcdf[(size_t)m * ldS + j] = 1.f;
}

__global__ void k_prepare_run(DeviceModel D, const double* __restrict__ mass, const double* __restrict__ Lsrc,
                              const double* __restrict__ epsref, double* cscale, double* eunit, ModelParams* mp,
                              double n_total, double qscale, int zero, const double* __restrict__ Ldust = nullptr,
                              float* qsdust = nullptr)
{
    const int ldS = D.ldS;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx == 0) { *D.ticket = 0u; if (zero) for (int c = 0; c < DIES_N_COUNTERS; c++) D.counters[c] = 0ull; }
    if (idx < D.n_models) {
        D.next_id[idx] = 0ull;
        ModelParams p = mp[idx];
        const double Le = p.has_ext ? Lsrc[2 * idx] : 0.0, Lp = p.has_point ? Lsrc[2 * idx + 1] : 0.0;
        const double Ld = Ldust ? Ldust[idx] : 0.0;          // TMC mode: the dust is a source of its own (R22)
        const double Lref = fmax(fmax(Le, Lp), Ld);
        p.qs_ext = Lref > 0 ? (float)(Le / Lref) : 0.f;
        p.qs_point = Lref > 0 ? (float)(Lp / Lref) : 0.f;
        if (qsdust) qsdust[idx] = Lref > 0 ? (float)(Ld / Lref) : 0.f;
        mp[idx] = p;
        eunit[idx] = Lref / n_total / qscale;
    }
    if (idx < D.n_models * ldS) {
        const int m = idx / ldS;
        const ModelParams p = mp[m];
        const double Le = p.has_ext ? Lsrc[2 * m] : 0.0, Lp = p.has_point ? Lsrc[2 * m + 1] : 0.0;
        const double eu = fmax(fmax(Le, Lp), Ldust ? Ldust[m] : 0.0) / n_total / qscale;
        const double ms = mass[idx];
        cscale[idx] = ms > 0.0 ? eu / (ms * *epsref) : 0.0;
        if (zero) D.A[(size_t)idx * kTallyStride] = 0ull;
    }
    if (zero && idx < D.n_models * D.K) D.esc[idx] = 0ull;
}

// temperatures from the tallies: eps = A e_unit / m, log-log interpolation in the (eps, T) table (L87; R6)
__global__ void k_finalize(DeviceModel D, const double* __restrict__ mass, const double* __restrict__ eunit,
                           const double* __restrict__ eps, const double* __restrict__ Tgrid, const ModelParams* mp,
                           double* T_out, double* Lesc_out, int* flags)
{
    const int N = D.N, K = D.K, nT = D.nT, ldS = D.ldS;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < D.n_models * K) {
        const unsigned long long v = D.esc[idx];
        if (v > (1ull << 62)) atomicOr(flags + 1, 1);
        Lesc_out[idx] = (double)v * eunit[idx / K];
    }
    if (idx < D.n_models * N) {
        const int m = idx / N, i = idx % N;
        const int j = i + mp[m].cav;
        const unsigned long long a = D.A[((size_t)m * ldS + j) * kTallyStride];
        if (a > (1ull << 62)) atomicOr(flags + 1, 1);
        const double ms = mass[(size_t)m * ldS + j];
        double T = 0.0;
        if (ms > 0.0) {
            const double e = (double)a * eunit[m] / ms;
            if (e < eps[0]) { T = Tgrid[0]; atomicAdd(&D.counters[DIES_C_T_CLAMP_LO], 1ull); }
            else if (e >= eps[nT - 1]) { T = Tgrid[nT - 1]; atomicAdd(&D.counters[DIES_C_T_CLAMP_HI], 1ull); }
            else {
                int lo = 0, hi = nT;      // first index with eps > e
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (eps[mid] > e) hi = mid; else lo = mid + 1; }
                const int t = lo - 1;
                const double f = (log(e) - log(eps[t])) / (log(eps[t + 1]) - log(eps[t]));
                T = exp(log(Tgrid[t]) + f * (log(Tgrid[t + 1]) - log(Tgrid[t])));
            }
        }
        T_out[idx] = T;
    }
}

__global__ void k_sum_escaped(DeviceModel D)
{
    unsigned long long s = 0;
    for (int x = threadIdx.x; x < D.n_models * D.K; x += blockDim.x) s += D.esc[x];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(&D.counters[DIES_C_ESCAPED_RAW], s);
}

__global__ void k_test_philox(uint32_t k0, uint32_t k1, unsigned long long first, uint32_t blk, uint32_t mi, int n,
                              uint32_t* words, float* uni)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= n) return;
    const unsigned long long id = first + x;
    uint32_t o[4];
    philox4x32_10(k0, k1, (uint32_t)id, (uint32_t)(id >> 32), blk, mi, o);
    for (int c = 0; c < 4; c++) { words[4 * x + c] = o[c]; uni[4 * x + c] = uniform24(o[c]); }
}

// ------------------------------------------------------------------ helpers
static int check_device()
{
    // (cudaGetDeviceProperties costs milliseconds; the compute capability is one attribute)
    int dev = 0, major = 0, minor = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(DIES_ECUDA, "no CUDA device: %s", cudaGetErrorString(e));
    CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CUDA_TRY(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    if (major != 10) return fail(DIES_ECUDA, "libdies is built for sm_100a only; device is sm_%d%d", major, minor);
    return DIES_OK;
}

// ------------------------------------------------------------------ launch tuning (include/dies.h: dies_tuning)
static const dies_tuning kTuningDefaults = {5, 4, 0, 32, (int32_t)kChunk, kFlyWarps * 32, 96, 20, 16, 32, kTallyStride};
static dies_tuning g_tuning = kTuningDefaults;
static std::mutex g_tuning_mutex;

static dies_tuning tuning()
{
    std::lock_guard<std::mutex> lock(g_tuning_mutex);
    return g_tuning;
}

extern "C" int dies_set_tuning(const dies_tuning* t)
{
    std::lock_guard<std::mutex> lock(g_tuning_mutex);
    if (!t) { g_tuning = kTuningDefaults; return DIES_OK; }
    dies_tuning n = g_tuning;
    struct { int32_t dies_tuning::*f; int lo, hi; const char* name; } spec[] = {
        {&dies_tuning::slots_uniform, 1, kMaxSlots, "slots_uniform"}, {&dies_tuning::slots, 1, kMaxSlots, "slots"},
        {&dies_tuning::visit, 1, 64, "visit"}, {&dies_tuning::min_ready, 1, 256, "min_ready"},
        {&dies_tuning::chunk, 32, 4096, "chunk"}, {&dies_tuning::pkg_per_block, 32, 1 << 20, "pkg_per_block"},
        {&dies_tuning::w_pool, 32, kMaxPool, "w_pool"}, {&dies_tuning::w_thr_hi, 1, 32, "w_thr_hi"},
        {&dies_tuning::w_thr_lo, 1, 32, "w_thr_lo"}, {&dies_tuning::w_min_ready, 1, kMaxPool, "w_min_ready"},
        {&dies_tuning::atom_stride, 1, 64, "atom_stride"}};
    for (auto& sp : spec) {
        const int v = t->*(sp.f);
        if (v == 0) continue;
        if (v < sp.lo || v > sp.hi) return fail(DIES_EINVAL, "dies_set_tuning: %s must be in [%d, %d]", sp.name, sp.lo, sp.hi);
        n.*(sp.f) = v;
    }
    n.w_pool &= ~7;
    g_tuning = n;
    return DIES_OK;
}

extern "C" int dies_get_tuning(dies_tuning* t)
{
    if (!t) return fail(DIES_EINVAL, "NULL argument");
    *t = tuning();
    return DIES_OK;
}

// pool slots per lane of dies_fly
// (with per-package quanta | with one quantum for all packages: 8 bytes less per slot, so a deeper pool fits)
static int fly_slots(bool uniform_q) { const dies_tuning t = tuning(); return uniform_q ? t.slots_uniform : t.slots; }

static size_t fly_smem(int N, int K, int nT, int M, bool trace, bool with_q, int logc)
{
    const int ldS = N + 1, ldT = 2 * ldS + 2;
    return plan_fly(K, nT, ldS, ldT, M, trace, with_q, logc).total;
}

// Launch shape of dies_fly for a model: 16 interleaved copies of the shell table when they fit beside a pool of at
// least 3 slots per lane, else one copy; the pool as deep as asked for, or as fits.
// The 227 KiB a block may opt in to cover its static shared memory too (s_ticket, s_cnt: 112 bytes in every tracker),
// so the plans get 227 KiB less a reserve for it; grant_smem checks that the reserve covers what the kernel declares.
constexpr size_t kStaticSmemReserve = 256;
constexpr size_t kFlySmemMax = 227 * 1024 - kStaticSmemReserve;
static bool fly_shape(int N, int K, int nT, int want_slots, bool trace, bool with_q, int* logc, int* slots)
{
    for (int lc = 4; lc >= 0; lc -= 4) {
        const int least = lc ? (want_slots < 3 ? want_slots : 3) : 1;
        for (int M = want_slots; M >= least; M--)
            if (fly_smem(N, K, nT, M, trace, with_q, lc) <= kFlySmemMax) { *logc = lc; *slots = M; return true; }
    }
    return false;
}

// shared memory of dies_track (weighted runs)
static size_t tracker_smem(int N, int K, int nT, int P, bool trace, bool with_q, bool wt = false)
{
    const int ldS = N + 1, ldT = 2 * ldS + 2;
    return plan_smem(K, nT, ldS, ldT, P, trace, with_q, wt).total;
}

// Dynamic shared memory a kernel may be launched with: raised per device and only upwards (a model that needs less
// must not lower it under a model that needs more), under a mutex (handles of different threads are independent).
enum { KF_FLY = 0 /* + mode + 2 trace + 4 (one table copy) */, KF_TRK0 = 8, KF_TRK1, KF_TRK0T, KF_TRK1T, KF_N };
static int fly_kernel(int mode, bool trace, int logc) { return KF_FLY + (mode == DIES_MODE_IRE ? 0 : 1) + (trace ? 2 : 0) + (logc ? 0 : 4); }
static const void* kernel_fn(int which)
{
    switch (which) {
    case 0: return (const void*)dies_fly<0, false, 4>;
    case 1: return (const void*)dies_fly<1, false, 4>;
    case 2: return (const void*)dies_fly<0, true, 4>;
    case 3: return (const void*)dies_fly<1, true, 4>;
    case 4: return (const void*)dies_fly<0, false, 0>;
    case 5: return (const void*)dies_fly<1, false, 0>;
    case 6: return (const void*)dies_fly<0, true, 0>;
    case 7: return (const void*)dies_fly<1, true, 0>;
    case KF_TRK0: return (const void*)dies_track<0, false, true>;
    case KF_TRK1: return (const void*)dies_track<1, false, true>;
    case KF_TRK0T: return (const void*)dies_track<0, true, true>;
    default: return (const void*)dies_track<1, true, true>;
    }
}
static void launch_fly(int which, int grid, size_t smem, cudaStream_t st, const DeviceModel& D, const RunParams& R,
                       const TraceParams& tp, const FlyPlan& fp)
{
    switch (which) {
    case 0: dies_fly<0, false, 4><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 1: dies_fly<1, false, 4><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 2: dies_fly<0, true, 4><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 3: dies_fly<1, true, 4><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 4: dies_fly<0, false, 0><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 5: dies_fly<1, false, 0><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    case 6: dies_fly<0, true, 0><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    default: dies_fly<1, true, 0><<<grid, kFlyBlock, smem, st>>>(D, R, tp, fp); break;
    }
}
static cudaError_t grant_smem(int which, size_t bytes)
{
    static std::mutex mu;
    static size_t granted[64][KF_N] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && bytes <= granted[dev][which]) return cudaSuccess;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, kernel_fn(which));
    if (e != cudaSuccess) return e;
    if (fa.sharedSizeBytes > kStaticSmemReserve) return cudaErrorInvalidConfiguration;   // (a build-time slip, not a user error)
    e = cudaFuncSetAttribute(kernel_fn(which), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && dev >= 0 && dev < 64) granted[dev][which] = bytes;
    return e;
}

extern "C" int dies_workspace_bytes(int n_shells, int n_freq, int n_T, int n_models, size_t* bytes)
{
    if (!bytes || n_shells < 1 || n_freq < 1 || n_T < 2 || n_models < 1) return fail(DIES_EINVAL, "bad sizes");
    *bytes = make_layout(n_shells, n_freq, n_T, n_models).total;
    return DIES_OK;
}

extern "C" int dies_device_info(int* n_sms, int* blocks_per_sm, int* threads_per_block)
{
    int rc = check_device();
    if (rc) return rc;
    int dev = 0, sms = 0, bps = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    bps = 1;                                     // dies_fly: one block of kFlyBlock threads per SM
    if (n_sms) *n_sms = sms;
    if (blocks_per_sm) *blocks_per_sm = bps;
    if (threads_per_block) *threads_per_block = kFlyBlock;
    return DIES_OK;
}

// ------------------------------------------------------------------ create
extern "C" int dies_create_batch(int n_models, int n_shells, const double* r_bounds, const double* rho, int n_freq,
                                 const double* freq, const double* kappa_abs, const double* kappa_sca,
                                 const double* g_hg, int n_T, const double* T_grid, const double* emis,
                                 void* workspace_dev, size_t workspace_bytes, dies_model** out)
{
    if (!out) return fail(DIES_EINVAL, "out is NULL");
    *out = nullptr;
    const int N = n_shells, K = n_freq, nT = n_T, M = n_models;
    if (N < 1 || K < 1 || nT < 2 || M < 1) return fail(DIES_EINVAL, "bad sizes");
    if (!r_bounds || !rho || !kappa_abs || !kappa_sca || !g_hg || !T_grid || !emis || !workspace_dev)
        return fail(DIES_EINVAL, "NULL argument");
    if (((uintptr_t)workspace_dev & 255) != 0) return fail(DIES_EINVAL, "workspace must be 256-byte aligned");
    for (int m = 0; m < M; m++) {
        const double* r = r_bounds + (size_t)m * (N + 1);
        if (!(r[0] >= 0.0)) return fail(DIES_EINVAL, "model %d: r_bounds[0] < 0", m);
        for (int i = 0; i < N; i++) {
            if (!(r[i + 1] > r[i])) return fail(DIES_EINVAL, "model %d: r_bounds not strictly ascending at %d", m, i);
            if (!(rho[(size_t)m * N + i] >= 0.0)) return fail(DIES_EINVAL, "model %d: rho[%d] < 0", m, i);
        }
    }
    double kref = 0.0;
    for (int k = 0; k < K; k++) {
        if (!(kappa_abs[k] >= 0.0) || !(kappa_sca[k] >= 0.0)) return fail(DIES_EINVAL, "negative opacity in bin %d", k);
        if (!(fabs(g_hg[k]) < 1.0)) return fail(DIES_EINVAL, "|g| >= 1 in bin %d", k);
        if (freq && k > 0 && !(freq[k] > freq[k - 1])) return fail(DIES_EINVAL, "freq not ascending at %d", k);
        kref = fmax(kref, kappa_abs[k] + kappa_sca[k]);
    }
    if (!(kref > 0.0)) kref = 1.0;
    for (int t = 1; t < nT; t++)
        if (!(T_grid[t] > T_grid[t - 1])) return fail(DIES_EINVAL, "T_grid not strictly ascending at %d", t);
    int rc = check_device();
    if (rc) return rc;
    const Layout L = make_layout(N, K, nT, M);
    if (workspace_bytes < L.total) return fail(DIES_ENOMEM, "workspace too small: %zu < %zu", workspace_bytes, L.total);
    // the smallest launch shapes of the two trackers must fit (the shapes of a run are chosen in dies_run)
    const int pool = tuning().w_pool;
    const size_t smem = fly_smem(N, K, nT, 1, false, true, 0);
    const size_t smem_trace = tracker_smem(N, K, nT, 32, true, true, true);
    if (smem_trace > 200 * 1024 || fly_smem(N, K, nT, 1, true, true, 0) > kFlySmemMax)
        return fail(DIES_EINVAL, "tables do not fit in shared memory (%zu bytes)", smem_trace);

    dies_model* m = new (std::nothrow) dies_model();
    if (!m) return fail(DIES_ENOMEM, "host allocation failed");
    m->N = N; m->K = K; m->nT = nT; m->M = M; m->ldS = N + 1;
    m->L = L; m->ws = (unsigned char*)workspace_dev;
    m->sources_set = m->fixed_set = m->ran = m->finalized = false;
    m->last_mode = DIES_MODE_IRE;
    m->done = m->n_total = 0; m->next_first = 0; m->shift = 24; m->model0 = 0; m->visit_auto = 8; m->stream = 0; m->launches = 0;
    m->L_point.assign(M, 0.0); m->has_ext.assign(M, 0); m->has_point.assign(M, 0);
    m->smem_bytes = smem; m->smem_trace_bytes = smem_trace; m->pool = pool; m->kref = kref;
    DeviceModel& D = m->D;
    D.N = N; D.K = K; D.nT = nT; D.n_models = M; D.ldS = N + 1; D.ldT = 2 * (N + 1) + 2;
    D.bintab = wsp<float4>(m, L.bintab); D.omega = wsp<float>(m, L.omega); D.epsgrid = wsp<float>(m, L.epsgrid);
    D.F = wsp<float>(m, L.F); D.guideF = wsp<unsigned short>(m, L.guideF); D.guideS = wsp<unsigned short>(m, L.guideS);
    D.stab = wsp<float2>(m, L.stab); D.stabW = wsp<float4>(m, L.stabW); D.cscale = wsp<double>(m, L.cscale);
    D.srccdf = wsp<float>(m, L.srccdf); D.mp = wsp<ModelParams>(m, L.mp); D.fixed_row = wsp<int>(m, L.fixed_row);
    D.A = wsp<unsigned long long>(m, L.A); D.esc = wsp<unsigned long long>(m, L.esc);
    D.next_id = wsp<unsigned long long>(m, L.next_id); D.counters = wsp<unsigned long long>(m, L.counters);
    D.ticket = wsp<unsigned int>(m, L.ticket);

#define TRY_OR_FREE(expr)                                                                                   \
    do {                                                                                                    \
        cudaError_t e_ = (expr);                                                                            \
        if (e_ != cudaSuccess) { delete m; return fail(DIES_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } \
    } while (0)
    TRY_OR_FREE(cudaMemsetAsync(m->ws, 0, L.total, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.emis, emis, (size_t)nT * K * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.Tgrid, T_grid, (size_t)nT * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.dustin, kappa_abs, (size_t)K * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.dustin + (size_t)K * 8, kappa_sca, (size_t)K * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.dustin + (size_t)2 * K * 8, g_hg, (size_t)K * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.rb, r_bounds, (size_t)M * (N + 1) * 8, cudaMemcpyHostToDevice, 0));
    TRY_OR_FREE(cudaMemcpyAsync(m->ws + L.rho, rho, (size_t)M * N * 8, cudaMemcpyHostToDevice, 0));
    int* flags = wsp<int>(m, L.flags);
    k_build_tables<<<(nT * 32 + 127) / 128, 128>>>(wsp<double>(m, L.emis), nT, K, wsp<double>(m, L.eps), wsp<float>(m, L.F), wsp<float>(m, L.G), flags);
    k_build_guide<<<(nT * kGuide + 255) / 256, 256>>>(wsp<float>(m, L.F), nT, K, wsp<unsigned short>(m, L.guideF));
    k_build_epsgrid<<<(nT + 127) / 128, 128>>>(wsp<double>(m, L.eps), nT, wsp<float>(m, L.epsgrid), wsp<double>(m, L.epsref), flags);
    k_build_dust<<<(K + 127) / 128, 128>>>(wsp<double>(m, L.dustin), K, kref, wsp<float4>(m, L.bintab), wsp<float>(m, L.omega));
    k_build_shells<<<(M * (2 * N + 4) + 127) / 128, 128>>>(wsp<double>(m, L.rb), wsp<double>(m, L.rho), N, M, kref,
                                                       wsp<float2>(m, L.stab), wsp<double>(m, L.mass), wsp<ModelParams>(m, L.mp));
    m->launches += 5;
    int hflags[2] = {0, 0};
    TRY_OR_FREE(cudaMemcpy(hflags, flags, sizeof(hflags), cudaMemcpyDeviceToHost));
    TRY_OR_FREE(cudaGetLastError());
    if (hflags[0] & 1) { delete m; return fail(DIES_EINVAL, "emis must be >= 0 and non-decreasing with T in every bin"); }
    if (hflags[0] & 2) { delete m; return fail(DIES_EINVAL, "row sums of emis must strictly increase with T"); }
    int dev = 0;
    TRY_OR_FREE(cudaGetDevice(&dev));
    TRY_OR_FREE(cudaDeviceGetAttribute(&m->n_sms, cudaDevAttrMultiProcessorCount, dev));
    m->blocks_per_sm = 1;
    m->grid_max = m->n_sms * m->blocks_per_sm;
#undef TRY_OR_FREE
    *out = m;
    return DIES_OK;
}

extern "C" int dies_create_model(int n_shells, const double* r_bounds, const double* rho, int n_freq, const double* freq,
                                 const double* kappa_abs, const double* kappa_sca, const double* g_hg, int n_T,
                                 const double* T_grid, const double* emis, void* workspace_dev, size_t workspace_bytes,
                                 dies_model** out)
{
    return dies_create_batch(1, n_shells, r_bounds, rho, n_freq, freq, kappa_abs, kappa_sca, g_hg, n_T, T_grid, emis,
                             workspace_dev, workspace_bytes, out);
}

extern "C" int dies_destroy(dies_model* m)
{
    if (!m) return DIES_OK;
    cudaStreamSynchronize(m->stream);
    delete m;
    return DIES_OK;
}

// ------------------------------------------------------------------ sources
extern "C" int dies_set_sources_batch(dies_model* m, const double* ext, const double* L_point, const double* point_w)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    const int K = m->K, M = m->M, N = m->N;
    std::vector<double> in((size_t)M * 2 * K, 0.0);
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    bool any = false;
    for (int i = 0; i < M; i++) {
        double J = 0.0, P = 0.0;
        if (ext) for (int k = 0; k < K; k++) {
            const double v = ext[(size_t)i * K + k];
            if (!(v >= 0.0)) return fail(DIES_EINVAL, "model %d: negative external intensity in bin %d", i, k);
            in[((size_t)i * 2) * K + k] = v; J += v;
        }
        const double Lp = L_point ? L_point[i] : 0.0;
        if (point_w && Lp > 0.0) for (int k = 0; k < K; k++) {
            const double v = point_w[(size_t)i * K + k];
            if (!(v >= 0.0)) return fail(DIES_EINVAL, "model %d: negative point-source weight in bin %d", i, k);
            in[((size_t)i * 2 + 1) * K + k] = v; P += v;
        }
        if (Lp < 0.0) return fail(DIES_EINVAL, "model %d: L_point < 0", i);
        m->has_ext[i] = J > 0.0; m->has_point[i] = (Lp > 0.0 && P > 0.0);
        m->L_point[i] = m->has_point[i] ? Lp : 0.0;
        any = any || m->has_ext[i] || m->has_point[i];
    }
    std::vector<double> Ls((size_t)2 * M, 0.0);
    for (int i = 0; i < M; i++) Ls[2 * i + 1] = m->L_point[i];
    CUDA_TRY(cudaMemcpy(m->ws + m->L.srcin, in.data(), in.size() * 8, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(m->ws + m->L.Lsrc, Ls.data(), Ls.size() * 8, cudaMemcpyHostToDevice));
    if ((size_t)K * 8 <= 40 * 1024)
        k_build_sources_staged<<<2 * M, 128, (size_t)K * 8>>>(wsp<double>(m, m->L.srcin), wsp<double>(m, m->L.rb), N, K, M,
                                                              wsp<float>(m, m->L.srccdf), wsp<double>(m, m->L.Lsrc),
                                                              wsp<ModelParams>(m, m->L.mp));
    else
        k_build_sources<<<(2 * M + 127) / 128, 128>>>(wsp<double>(m, m->L.srcin), wsp<double>(m, m->L.rb), N, K, M,
                                                      wsp<float>(m, m->L.srccdf), wsp<double>(m, m->L.Lsrc),
                                                      wsp<ModelParams>(m, m->L.mp));
    k_build_guide<<<(2 * M * kGuide + 255) / 256, 256>>>(wsp<float>(m, m->L.srccdf), 2 * M, K,
                                                        wsp<unsigned short>(m, m->L.guideS));
    m->launches += 2;
    CUDA_TRY(cudaGetLastError());
    // the tables are built on the legacy default stream; dies_run may use any stream (also a non-blocking one)
    CUDA_TRY(cudaDeviceSynchronize());
    m->sources_set = any;
    m->ran = false; m->done = 0;
    return DIES_OK;
}

extern "C" int dies_set_sources(dies_model* m, const double* ext, double L_point, const double* point_w)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    if (m->M != 1) return fail(DIES_EINVAL, "use dies_set_sources_batch for a batch handle");
    return dies_set_sources_batch(m, ext, &L_point, point_w);
}

extern "C" int dies_set_fixed_temperature(dies_model* m, const double* T, int n)
{
    if (!m || !T) return fail(DIES_EINVAL, "NULL argument");
    if (n != m->M * m->N) return fail(DIES_EINVAL, "n must be n_models*n_shells = %d", m->M * m->N);
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    CUDA_TRY(cudaMemcpy(m->ws + m->L.Tfix, T, (size_t)n * 8, cudaMemcpyHostToDevice));
    k_fixed_rows<<<(n + 127) / 128, 128>>>(wsp<double>(m, m->L.Tfix), wsp<double>(m, m->L.Tgrid), m->nT, m->N, m->M,
                                           wsp<ModelParams>(m, m->L.mp), wsp<int>(m, m->L.fixed_row));
    m->launches += 1;
    CUDA_TRY(cudaDeviceSynchronize());
    m->fixed_set = true;
    return DIES_OK;
}

// ------------------------------------------------------------------ run

constexpr unsigned kTmcSmemMax = 200 * 1024;     // dynamic shared memory dies_tmc is allowed
static int fill_run_params(dies_model* m, uint64_t n_packages, uint64_t seed, const dies_run_opts* o, RunParams* R,
                           int* mode, int* accumulate, int* shift, uint64_t* n_total)
{
    dies_run_opts d = {0.5, 0, DIES_MODE_IRE, 0, 24, 0, 1.0, 0.0, 1.0, 0.0, 0.0, 0, 0};
    if (o) d = *o;
    if (d.k_A == 0.0) d.k_A = 1.0;
    if (d.k_S == 0.0) d.k_S = 1.0;
    if (!(d.k_A > 0.0) || !(d.k_S > 0.0) || !(d.k_A_dilute >= 0.0)) return fail(DIES_EINVAL, "k_A, k_S must be > 0 and k_A_dilute >= 0");
    if (!(fabs(d.g_E) < 1.0) || !(fabs(d.g_S) < 1.0)) return fail(DIES_EINVAL, "|g_E|, |g_S| must be < 1");
    const bool weighted = d.k_A != 1.0 || d.k_S != 1.0 || d.k_A_dilute > 0.0 || d.g_E != 0.0 || d.use_g_S != 0 ||
                          d.reemit_in_cell != 0;
    if (weighted && d.ffi) return fail(DIES_EINVAL, "free-path / directional weighting and forced first interaction are alternatives, not combined");
    if (!(d.k_bg > 0.0) || d.k_bg > 1.0) return fail(DIES_EINVAL, "k_bg must be in (0, 1]");
    if (d.mode != DIES_MODE_IRE && d.mode != DIES_MODE_FIXED_T && d.mode != DIES_MODE_TMC) return fail(DIES_EINVAL, "bad mode");
    if (d.mode == DIES_MODE_TMC && (weighted || d.ffi || d.k_bg != 0.5 || d.accumulate || (d.n_total && d.n_total != n_packages)))
        return fail(DIES_EINVAL, "a TMC iteration is one plain run: no weighting, no forced first interaction, no accumulate");
    if (d.fixed_shift == 0) d.fixed_shift = 24;
    if (d.fixed_shift < 1 || d.fixed_shift > 30) return fail(DIES_EINVAL, "fixed_shift must be in [1, 30]");
    if (d.n_total == 0) d.n_total = n_packages;
    if (d.mode == DIES_MODE_FIXED_T && !m->fixed_set) return fail(DIES_ESTATE, "fixed-T mode needs dies_set_fixed_temperature");
    if (d.mode == DIES_MODE_TMC) {
        // (checked here, before dies_run writes to the handle: a rejected call must leave dies_seek, n_total and the
        // stream of the handle as they were)
        if (d.fixed_shift > 24) return fail(DIES_EINVAL, "TMC mode keeps package quanta in 32 bits: fixed_shift <= 24");
        if (plan_tmc(m->K, m->ldS, m->D.ldT).total > kTmcSmemMax) return fail(DIES_EINVAL, "tables do not fit in shared memory");
    }
    *mode = d.mode; *accumulate = d.accumulate; *shift = d.fixed_shift; *n_total = d.n_total;
    int two = 0;
    for (int i = 0; i < m->M; i++) two |= (m->has_ext[i] && m->has_point[i]);
    R->n_run = n_packages; R->n_total = d.n_total; R->id_base = 0;
    R->key0 = (uint32_t)seed; R->key1 = (uint32_t)(seed >> 32);
    R->model0 = m->model0;
    for (int r = 0; r < 10; r++) { R->rk[2 * r] = R->key0 + (uint32_t)r * 0x9E3779B9u; R->rk[2 * r + 1] = R->key1 + (uint32_t)r * 0xBB67AE85u; }
    R->k_bg = (float)d.k_bg; R->ffi = d.ffi ? 1 : 0;
    R->uniform_q = (d.k_bg == 0.5 && !d.ffi && !two && !weighted) ? 1 : 0;
    R->weighted = weighted ? 1 : 0;
    R->k_S = (float)d.k_S; R->k_A = d.k_A; R->k_A_dilute = d.k_A_dilute;
    R->g_E = (float)d.g_E; R->g_S = (float)d.g_S; R->use_gS = d.use_g_S ? 1 : 0;
    R->reemit_cell = d.reemit_in_cell ? 1 : 0;
    R->qscale = (float)(1u << d.fixed_shift);
    const dies_tuning tn = tuning();
    R->pool = tn.w_pool;
    R->thr_hi = tn.w_thr_hi; R->thr_lo = tn.w_thr_lo; R->min_ready = tn.w_min_ready;
    R->slots = fly_slots(R->uniform_q != 0);
    R->visit = tn.visit > 0 ? tn.visit : m->visit_auto;
    if (!weighted) R->min_ready = tn.min_ready;
    R->n_tickets = 0; R->parts = 1;
    return DIES_OK;
}

extern "C" int dies_run(dies_model* m, uint64_t n_packages, uint64_t seed, const dies_run_opts* opts, void* cuda_stream)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    if (!m->sources_set) return fail(DIES_ESTATE, "dies_run before dies_set_sources");
    if (n_packages == 0) return fail(DIES_EINVAL, "n_packages is 0");
    RunParams R;
    int mode, accumulate, shift; uint64_t n_total;
    int rc = fill_run_params(m, n_packages, seed, opts, &R, &mode, &accumulate, &shift, &n_total);
    if (rc) return rc;
    if (accumulate && m->ran) {
        if (n_total != m->n_total || shift != m->shift) return fail(DIES_ESTATE, "accumulate needs the same n_total and fixed_shift");
        // the raw unit of a TMC run includes the dust luminosity: its tallies cannot be continued by another mode
        if (m->last_mode == DIES_MODE_TMC) return fail(DIES_ESTATE, "accumulate after a TMC run: the tallies are in the TMC energy unit");
    } else {
        accumulate = 0;
        m->done = m->next_first;
    }
    m->next_first = 0;
    if (m->done + n_packages > n_total) return fail(DIES_EINVAL, "more packages than n_total");
    R.id_base = m->done;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (m->ran && st != m->stream) CUDA_TRY(cudaStreamSynchronize(m->stream));
    m->stream = st;
    m->n_total = n_total; m->shift = shift;

    if (mode == DIES_MODE_TMC) {
        // one iteration of the traditional Monte Carlo (dies_tmc.cuh): the dust emits what the run before left in it
        const TmcPlan tpn = plan_tmc(m->K, m->ldS, m->D.ldT);      // (size and fixed_shift checked in fill_run_params)
        static std::mutex mu;
        {
            std::lock_guard<std::mutex> lock(mu);
            CUDA_TRY(cudaFuncSetAttribute(dies_tmc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTmcSmemMax));
        }
        int bps = 0;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, dies_tmc, kBlock, tpn.total));
        if (bps < 1) return fail(DIES_ECUDA, "tracker does not fit on an SM");
        const int grid = m->n_sms * bps;
        R.chunk = 32u * 8u;
        if (m->M == 1) { R.parts = grid; R.n_tickets = grid; }
        else { R.parts = (8 * grid + m->M - 1) / m->M; if (R.parts < 1) R.parts = 1; R.n_tickets = m->M * R.parts; }
        k_tmc_prepare<<<(m->M + 63) / 64, 64, 0, st>>>(m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.eunit),
                                                      wsp<double>(m, m->L.eps), m->ran ? 1 : 0, wsp<double>(m, m->L.epscur),
                                                      wsp<float>(m, m->L.cellcdf), wsp<int>(m, m->L.tmcrow),
                                                      wsp<float>(m, m->L.tmcmix), wsp<double>(m, m->L.Ldust));
        const int prep = m->M * (m->K > m->ldS ? m->K : m->ldS);
        k_prepare_run<<<(prep + 255) / 256, 256, 0, st>>>(m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.Lsrc),
                                                        wsp<double>(m, m->L.epsref), wsp<double>(m, m->L.cscale),
                                                        wsp<double>(m, m->L.eunit), wsp<ModelParams>(m, m->L.mp),
                                                        (double)n_total, (double)R.qscale, 1, wsp<double>(m, m->L.Ldust),
                                                        wsp<float>(m, m->L.qsdust));
        const TmcModel Tm = {wsp<float>(m, m->L.G), wsp<float>(m, m->L.cellcdf), wsp<int>(m, m->L.tmcrow),
                             wsp<float>(m, m->L.tmcmix), wsp<float>(m, m->L.qsdust)};
        dies_tmc<<<grid, kBlock, tpn.total, st>>>(m->D, R, Tm, tpn);
        m->launches += 3;
        CUDA_TRY(cudaGetLastError());
        m->done += n_packages;
        m->ran = true;
        m->last_mode = DIES_MODE_TMC;
        m->finalized = false;
        return DIES_OK;
    }

    // launch shape: shared memory of this run's pool, persistent blocks (as many as fit on an SM), fewer for tiny runs
    const bool wt = R.weighted != 0;
    const dies_tuning tn = tuning();
    int logc = 0;
    if (!wt && !fly_shape(m->N, m->K, m->nT, R.slots, false, !R.uniform_q, &logc, &R.slots))
        return fail(DIES_ECUDA, "tracker does not fit on an SM");
    const int kf = wt ? (mode == DIES_MODE_IRE ? KF_TRK0 : KF_TRK1) : fly_kernel(mode, false, logc);
    const FlyPlan fp = plan_fly(m->K, m->nT, m->ldS, m->D.ldT, R.slots, false, !R.uniform_q, logc);
    const size_t smem_launch = wt ? tracker_smem(m->N, m->K, m->nT, R.pool, false, !R.uniform_q, true) : fp.total;
    const int threads = wt ? kBlock : kFlyBlock, warps = threads / 32;
    CUDA_TRY(grant_smem(kf, smem_launch));
    int bps = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel_fn(kf), threads, smem_launch));
    if (bps < 1) return fail(DIES_ECUDA, "tracker does not fit on an SM");
    const int grid_max = m->n_sms * bps;
    unsigned long long ids = 0;
    for (int i = 0; i < m->M; i++) ids += n_packages * (unsigned long long)(m->has_ext[i] + m->has_point[i]);
    // small runs: 32 packages per warp and chunks to match, so that every SM takes part; large runs: the whole grid
    const unsigned long long per_b = wt ? (unsigned long long)(kWarps * 32) : (unsigned long long)tn.pkg_per_block;
    unsigned long long want = (ids + per_b - 1) / per_b;
    int grid = (int)(want < 1 ? 1 : (want > (unsigned long long)grid_max ? grid_max : want));
    {
        const unsigned long long per_warp = ids / ((unsigned long long)grid * warps * (unsigned long long)m->M) ;
        const unsigned long long cmax = (unsigned long long)tn.chunk;
        R.chunk = (unsigned)(per_warp < 32 ? 32 : (per_warp > cmax ? cmax : per_warp));
    }
    if (m->M == 1) { R.parts = grid; R.n_tickets = grid; }
    else { R.parts = (8 * grid + m->M - 1) / m->M; if (R.parts < 1) R.parts = 1; R.n_tickets = m->M * R.parts; }

    const int prep = m->M * (m->K > m->ldS ? m->K : m->ldS);
    k_prepare_run<<<(prep + 255) / 256, 256, 0, st>>>(m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.Lsrc),
                                                    wsp<double>(m, m->L.epsref), wsp<double>(m, m->L.cscale),
                                                    wsp<double>(m, m->L.eunit), wsp<ModelParams>(m, m->L.mp),
                                                    (double)n_total, (double)R.qscale, accumulate ? 0 : 1);
    TraceParams tp = {0, 0, 0, nullptr, 0, nullptr, nullptr};
    if (wt) {
        // shell table with the weighting factors of this run
        const int nw = m->M * (2 * m->ldS + 2);
        k_build_wshells<<<(nw + 127) / 128, 128, 0, st>>>(wsp<double>(m, m->L.rb), wsp<double>(m, m->L.rho), m->N, m->M, m->kref,
                                                       R.k_A, R.k_A_dilute, wsp<float4>(m, m->L.stabW));
        m->launches += 1;
        if (mode == DIES_MODE_IRE) dies_track<0, false, true><<<grid, kBlock, smem_launch, st>>>(m->D, R, tp);
        else dies_track<1, false, true><<<grid, kBlock, smem_launch, st>>>(m->D, R, tp);
    } else {
        launch_fly(kf, grid, smem_launch, st, m->D, R, tp, fp);
    }
    m->launches += 2;
    CUDA_TRY(cudaGetLastError());
    m->done += n_packages;
    m->ran = true;
    m->last_mode = mode;
    m->finalized = false;
    return DIES_OK;
}

extern "C" int dies_seek(dies_model* m, uint64_t first_id)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    m->next_first = first_id;
    return DIES_OK;
}

extern "C" int dies_set_model_offset(dies_model* m, uint32_t first_model)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    if ((uint64_t)first_model + (uint64_t)m->M > 0xffffffffull) return fail(DIES_EINVAL, "model index beyond 2^32");
    m->model0 = first_model;
    return DIES_OK;
}

extern "C" int dies_run_batch(dies_model* m, uint64_t n, uint64_t seed, const dies_run_opts* opts, void* cuda_stream)
{
    return dies_run(m, n, seed, opts, cuda_stream);
}

// ------------------------------------------------------------------ getters
static int finalize(dies_model* m)
{
    if (!m->ran) return fail(DIES_ESTATE, "no run yet");
    if (m->finalized) return DIES_OK;            // nothing ran since the last read-out
    const int n = m->M * (m->K > m->N ? m->K : m->N);
    int* flags = wsp<int>(m, m->L.flags);
    CUDA_TRY(cudaMemsetAsync(flags, 0, 16, m->stream));
    // the derived counters ESCAPED_RAW, T_CLAMP_LO, T_CLAMP_HI are recomputed by every finalisation
    CUDA_TRY(cudaMemsetAsync(m->ws + m->L.counters + DIES_C_ESCAPED_RAW * 8, 0, 3 * 8, m->stream));
    k_finalize<<<(n + 255) / 256, 256, 0, m->stream>>>(m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.eunit),
                                                     wsp<double>(m, m->L.eps), wsp<double>(m, m->L.Tgrid),
                                                     wsp<ModelParams>(m, m->L.mp), wsp<double>(m, m->L.T_out),
                                                     wsp<double>(m, m->L.Lesc_out), flags);
    k_sum_escaped<<<1, 256, 0, m->stream>>>(m->D);
    m->launches += 2;
    int hf[2];
    unsigned long long hc[DIES_C_ABSORPTIONS + 1];
    CUDA_TRY(cudaMemcpyAsync(hf, flags, sizeof(hf), cudaMemcpyDeviceToHost, m->stream));
    CUDA_TRY(cudaMemcpyAsync(hc, m->ws + m->L.counters, sizeof(hc), cudaMemcpyDeviceToHost, m->stream));
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    CUDA_TRY(cudaGetLastError());
    if (hf[1]) return fail(DIES_EOVERFLOW, "a tally exceeded 2^62");
    {
        // launch tuning of the next runs of this model (dies_tuning.visit = 0): a crossing phase of dies_fly lasts
        // about two mean flights (a flight: the crossings between two events of a package).  Order of work only.
        const double flights = (double)(hc[DIES_C_PACKAGES] + hc[DIES_C_SCATTERINGS] + hc[DIES_C_ABSORPTIONS]);
        if (flights > 0.0) {
            const double steps = 2.0 * (double)hc[DIES_C_CROSSINGS] / flights;
            int v = (int)(steps / kSteps + 0.999);
            m->visit_auto = v < 2 ? 2 : (v > 8 ? 8 : v);
        }
    }
    m->finalized = true;
    return DIES_OK;
}

extern "C" int dies_get_temperature(dies_model* m, double* T, int n)
{
    if (!m || !T) return fail(DIES_EINVAL, "NULL argument");
    if (n != m->M * m->N) return fail(DIES_EINVAL, "n must be n_models*n_shells = %d", m->M * m->N);
    int rc = finalize(m);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpy(T, m->ws + m->L.T_out, (size_t)n * 8, cudaMemcpyDeviceToHost));
    return DIES_OK;
}

extern "C" int dies_get_escape_spectrum(dies_model* m, double* Lesc, int n)
{
    if (!m || !Lesc) return fail(DIES_EINVAL, "NULL argument");
    if (n != m->M * m->K) return fail(DIES_EINVAL, "n must be n_models*n_freq = %d", m->M * m->K);
    int rc = finalize(m);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpy(Lesc, m->ws + m->L.Lesc_out, (size_t)n * 8, cudaMemcpyDeviceToHost));
    return DIES_OK;
}

extern "C" int dies_get_absorbed(dies_model* m, int64_t* raw, double* energy_per_raw_unit, int n)
{
    if (!m || !raw) return fail(DIES_EINVAL, "NULL argument");
    if (n != m->M * m->N) return fail(DIES_EINVAL, "n must be n_models*n_shells = %d", m->M * m->N);
    if (!m->ran) return fail(DIES_ESTATE, "no run yet");
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    std::vector<unsigned long long> a((size_t)m->M * m->ldS);
    std::vector<ModelParams> mp(m->M);
    // the tallies are kTallyStride words apart on the device
    CUDA_TRY(cudaMemcpy2D(a.data(), 8, m->ws + m->L.A, (size_t)kTallyStride * 8, 8, a.size(), cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(mp.data(), m->ws + m->L.mp, mp.size() * sizeof(ModelParams), cudaMemcpyDeviceToHost));
    for (int i = 0; i < m->M; i++)
        for (int s = 0; s < m->N; s++) {
            const unsigned long long v = a[(size_t)i * m->ldS + s + mp[i].cav];
            if (v > (1ull << 62)) return fail(DIES_EOVERFLOW, "a tally exceeded 2^62");
            raw[(size_t)i * m->N + s] = (int64_t)v;
        }
    if (energy_per_raw_unit) CUDA_TRY(cudaMemcpy(energy_per_raw_unit, m->ws + m->L.eunit, (size_t)m->M * 8, cudaMemcpyDeviceToHost));
    return DIES_OK;
}

extern "C" int dies_get_counters(dies_model* m, uint64_t* c, int n)
{
    if (!m || !c) return fail(DIES_EINVAL, "NULL argument");
    if (n != DIES_N_COUNTERS) return fail(DIES_EINVAL, "n must be DIES_N_COUNTERS = %d", (int)DIES_N_COUNTERS);
    int rc = finalize(m);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpy(c, m->ws + m->L.counters, (size_t)n * 8, cudaMemcpyDeviceToHost));
    c[DIES_C_KERNEL_LAUNCHES] = m->launches;
    return DIES_OK;
}

extern "C" int dies_get_tables(dies_model* m, double* eps, float* F)
{
    if (!m) return fail(DIES_EINVAL, "model is NULL");
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    if (eps) CUDA_TRY(cudaMemcpy(eps, m->ws + m->L.eps, (size_t)m->nT * 8, cudaMemcpyDeviceToHost));
    if (F) CUDA_TRY(cudaMemcpy(F, m->ws + m->L.F, (size_t)m->nT * m->K * 4, cudaMemcpyDeviceToHost));
    return DIES_OK;
}

// ------------------------------------------------------------------ trace / tests
extern "C" int dies_trace_packages(dies_model* m, int model_index, uint64_t first_id, int count, uint64_t n_total,
                                   uint64_t seed, const dies_run_opts* opts, int32_t* events, int max_events,
                                   int32_t* n_events)
{
    if (!m || !events || !n_events) return fail(DIES_EINVAL, "NULL argument");
    if (!m->sources_set) return fail(DIES_ESTATE, "trace before dies_set_sources");
    if (model_index < 0 || model_index >= m->M || count < 1 || max_events < 1 || n_total == 0)
        return fail(DIES_EINVAL, "bad trace arguments");
    RunParams R;
    int mode, accumulate, shift; uint64_t nt;
    dies_run_opts o = {0.5, 0, DIES_MODE_FIXED_T, 0, 24, n_total, 1.0, 0.0, 1.0, 0.0, 0.0, 0, 0};
    if (opts) o = *opts;
    o.n_total = n_total;
    int rc = fill_run_params(m, 1, seed, &o, &R, &mode, &accumulate, &shift, &nt);
    if (rc) return rc;
    if (mode == DIES_MODE_TMC) return fail(DIES_EINVAL, "traces replay IRE or fixed-temperature packages, not a TMC iteration");
    if (mode == DIES_MODE_IRE && (!m->ran || nt != m->n_total || shift != m->shift || m->last_mode == DIES_MODE_TMC))
        return fail(DIES_ESTATE, "IRE-mode trace replays against the tallies of an IRE or fixed-temperature run with the same n_total");
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    if (!m->ran) {
        // energy scales are set per run; a trace before any run sets them for n_total
        k_prepare_run<<<(m->M * (m->K > m->ldS ? m->K : m->ldS) + 255) / 256, 256>>>(
            m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.Lsrc), wsp<double>(m, m->L.epsref),
            wsp<double>(m, m->L.cscale), wsp<double>(m, m->L.eunit), wsp<ModelParams>(m, m->L.mp), (double)nt,
            (double)R.qscale, 1);
        m->launches += 1;
    }
    R.n_run = nt; R.id_base = 0;
    R.uniform_q = 0;                                       // the trace kernels keep the quantum per package
    R.slots = fly_slots(false);
    R.chunk = 32;
    int32_t *d_ev = nullptr, *d_n = nullptr;
    CUDA_TRY(cudaMalloc(&d_ev, (size_t)count * max_events * 16));
    // n_events (count ints) followed by the 64-bit counter the traced package indices are taken from
    const size_t n_bytes = (((size_t)count * 4 + 7) & ~(size_t)7) + 8;
    if (cudaMalloc(&d_n, n_bytes) != cudaSuccess) { cudaFree(d_ev); return fail(DIES_ECUDA, "cudaMalloc failed"); }
    cudaMemset(d_n, 0, n_bytes);
    TraceParams tp = {model_index, first_id, count, d_ev, max_events, d_n,
                      reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(d_n) + n_bytes - 8)};
    cudaError_t ge = cudaSuccess;
    if (R.weighted) {
        int grid = (count + kBlock - 1) / kBlock;
        if (grid > 4 * m->n_sms) grid = 4 * m->n_sms;
        const int nw = m->M * (2 * m->ldS + 2);
        k_build_wshells<<<(nw + 127) / 128, 128>>>(wsp<double>(m, m->L.rb), wsp<double>(m, m->L.rho), m->N, m->M, m->kref,
                                                  R.k_A, R.k_A_dilute, wsp<float4>(m, m->L.stabW));
        m->launches += 1;
        const size_t sm = tracker_smem(m->N, m->K, m->nT, R.pool, true, true, true);
        ge = grant_smem(mode == DIES_MODE_IRE ? KF_TRK0T : KF_TRK1T, sm);
        if (ge == cudaSuccess) {
            if (mode == DIES_MODE_IRE) dies_track<0, true, true><<<grid, kBlock, sm>>>(m->D, R, tp);
            else dies_track<1, true, true><<<grid, kBlock, sm>>>(m->D, R, tp);
        }
    } else {
        int grid = (count + kFlyBlock - 1) / kFlyBlock;
        if (grid > m->grid_max) grid = m->grid_max;
        int logc = 0;
        if (!fly_shape(m->N, m->K, m->nT, R.slots, true, true, &logc, &R.slots)) {
            cudaFree(d_ev); cudaFree(d_n);
            return fail(DIES_ECUDA, "tracker does not fit on an SM");
        }
        const FlyPlan fp = plan_fly(m->K, m->nT, m->ldS, m->D.ldT, R.slots, true, true, logc);
        const int kf = fly_kernel(mode, true, logc);
        ge = grant_smem(kf, fp.total);
        if (ge == cudaSuccess) launch_fly(kf, grid, fp.total, 0, m->D, R, tp, fp);
    }
    if (ge != cudaSuccess) { cudaFree(d_ev); cudaFree(d_n); return fail(DIES_ECUDA, "trace: %s", cudaGetErrorString(ge)); }
    m->launches += 1;
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(events, d_ev, (size_t)count * max_events * 16, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(n_events, d_n, (size_t)count * 4, cudaMemcpyDeviceToHost);
    cudaFree(d_ev); cudaFree(d_n);
    if (e != cudaSuccess) return fail(DIES_ECUDA, "trace: %s", cudaGetErrorString(e));
    return DIES_OK;
}

extern "C" int dies_trace_package(dies_model* m, uint64_t package_id, uint64_t n_total, uint64_t seed,
                                  const dies_run_opts* opts, int32_t* events, int max_events, int32_t* n_events)
{
    return dies_trace_packages(m, 0, package_id, 1, n_total, seed, opts, events, max_events, n_events);
}

// ------------------------------------------------------------------ trace without any device allocation
// dies_trace_packages needs device scratch beyond the model's workspace: the event lists (count x max_events x 16
// bytes), the per-package event counts and the 64-bit counter the traced package indices are handed out from.  It
// gets them from cudaMalloc / cudaFree.  dies_trace_packages_static keeps the same scratch in the array below, which
// is part of the library image: every GPU that loads libdies.so holds these ~1.02 MiB until the process exits, and
// nothing is allocated or freed at call time.
//
// g_trace_scratch is a DEVICE symbol.  In host code its name is only a host-side stand-in and not a device address, so
// the host never passes `g_trace_scratch` itself to a kernel: trace_scratch() asks the runtime for the address once
// per device, with that device current, and hands that pointer on.
constexpr size_t kTraceStaticEvBytes = (size_t)DIES_TRACE_STATIC_MAX_EVENTS * 16;          // event quadruples
constexpr size_t kTraceStaticNBytes = (size_t)DIES_TRACE_STATIC_MAX_PACKAGES * 4;          // n_events
constexpr size_t kTraceStaticBytes = kTraceStaticEvBytes + kTraceStaticNBytes + 256;       // + the package counter
static __device__ __align__(256) unsigned char g_trace_scratch[kTraceStaticBytes];

static int trace_scratch(unsigned char** out)
{
    static std::mutex mu;
    static unsigned char* addr[64] = {};          // per device ordinal; the address differs from GPU to GPU
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(DIES_ECUDA, "device ordinal %d beyond the 64 this entry point keeps scratch addresses for", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_trace_scratch));
        if (!p) return fail(DIES_ECUDA, "cudaGetSymbolAddress gave no address for the trace scratch");
        addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = addr[dev];
    return DIES_OK;
}

extern "C" int dies_trace_packages_static(dies_model* m, int model_index, uint64_t first_id, int count, uint64_t n_total,
                                          uint64_t seed, const dies_run_opts* opts, int32_t* events, int max_events,
                                          int32_t* n_events)
{
    if (!m || !events || !n_events) return fail(DIES_EINVAL, "NULL argument");
    if (!m->sources_set) return fail(DIES_ESTATE, "trace before dies_set_sources");
    if (model_index < 0 || model_index >= m->M || count < 1 || max_events < 1 || n_total == 0)
        return fail(DIES_EINVAL, "bad trace arguments");
    if (count > DIES_TRACE_STATIC_MAX_PACKAGES)
        return fail(DIES_EINVAL, "dies_trace_packages_static: count %d exceeds DIES_TRACE_STATIC_MAX_PACKAGES = %d "
                    "(split the id range, or use dies_trace_packages, which allocates)", count, DIES_TRACE_STATIC_MAX_PACKAGES);
    if ((unsigned long long)count * (unsigned long long)max_events > (unsigned long long)DIES_TRACE_STATIC_MAX_EVENTS)
        return fail(DIES_EINVAL, "dies_trace_packages_static: count * max_events = %llu exceeds DIES_TRACE_STATIC_MAX_EVENTS = %d "
                    "(split the id range, or use dies_trace_packages, which allocates)",
                    (unsigned long long)count * (unsigned long long)max_events, DIES_TRACE_STATIC_MAX_EVENTS);
    RunParams R;
    int mode, accumulate, shift; uint64_t nt;
    dies_run_opts o = {0.5, 0, DIES_MODE_FIXED_T, 0, 24, n_total, 1.0, 0.0, 1.0, 0.0, 0.0, 0, 0};
    if (opts) o = *opts;
    o.n_total = n_total;
    int rc = fill_run_params(m, 1, seed, &o, &R, &mode, &accumulate, &shift, &nt);
    if (rc) return rc;
    if (mode == DIES_MODE_TMC) return fail(DIES_EINVAL, "traces replay IRE or fixed-temperature packages, not a TMC iteration");
    if (mode == DIES_MODE_IRE && (!m->ran || nt != m->n_total || shift != m->shift || m->last_mode == DIES_MODE_TMC))
        return fail(DIES_ESTATE, "IRE-mode trace replays against the tallies of an IRE or fixed-temperature run with the same n_total");
    unsigned char* scratch = nullptr;             // device address of g_trace_scratch on the current GPU
    rc = trace_scratch(&scratch);
    if (rc) return rc;
    CUDA_TRY(cudaStreamSynchronize(m->stream));
    if (!m->ran) {
        // energy scales are set per run; a trace before any run sets them for n_total
        k_prepare_run<<<(m->M * (m->K > m->ldS ? m->K : m->ldS) + 255) / 256, 256>>>(
            m->D, wsp<double>(m, m->L.mass), wsp<double>(m, m->L.Lsrc), wsp<double>(m, m->L.epsref),
            wsp<double>(m, m->L.cscale), wsp<double>(m, m->L.eunit), wsp<ModelParams>(m, m->L.mp), (double)nt,
            (double)R.qscale, 1);
        m->launches += 1;
    }
    R.n_run = nt; R.id_base = 0;
    R.uniform_q = 0;                                       // the trace kernels keep the quantum per package
    R.slots = fly_slots(false);
    R.chunk = 32;
    // The array still holds what the last call (of any handle, any thread) left in it.  The event counts and the
    // package counter must start at zero; the event lists of this call are cleared too, so that entries past a
    // package's n_events read as zeros rather than as another call's events.
    int32_t* const d_ev = reinterpret_cast<int32_t*>(scratch);
    int32_t* const d_n = reinterpret_cast<int32_t*>(scratch + kTraceStaticEvBytes);
    unsigned long long* const d_counter = reinterpret_cast<unsigned long long*>(scratch + kTraceStaticEvBytes + kTraceStaticNBytes);
    CUDA_TRY(cudaMemsetAsync(d_ev, 0, (size_t)count * max_events * 16, 0));
    CUDA_TRY(cudaMemsetAsync(d_n, 0, kTraceStaticNBytes + 8, 0));
    TraceParams tp = {model_index, first_id, count, d_ev, max_events, d_n, d_counter};
    cudaError_t ge = cudaSuccess;
    if (R.weighted) {
        int grid = (count + kBlock - 1) / kBlock;
        if (grid > 4 * m->n_sms) grid = 4 * m->n_sms;
        const int nw = m->M * (2 * m->ldS + 2);
        k_build_wshells<<<(nw + 127) / 128, 128>>>(wsp<double>(m, m->L.rb), wsp<double>(m, m->L.rho), m->N, m->M, m->kref,
                                                  R.k_A, R.k_A_dilute, wsp<float4>(m, m->L.stabW));
        m->launches += 1;
        const size_t sm = tracker_smem(m->N, m->K, m->nT, R.pool, true, true, true);
        ge = grant_smem(mode == DIES_MODE_IRE ? KF_TRK0T : KF_TRK1T, sm);
        if (ge == cudaSuccess) {
            if (mode == DIES_MODE_IRE) dies_track<0, true, true><<<grid, kBlock, sm>>>(m->D, R, tp);
            else dies_track<1, true, true><<<grid, kBlock, sm>>>(m->D, R, tp);
        }
    } else {
        int grid = (count + kFlyBlock - 1) / kFlyBlock;
        if (grid > m->grid_max) grid = m->grid_max;
        int logc = 0;
        if (!fly_shape(m->N, m->K, m->nT, R.slots, true, true, &logc, &R.slots))
            return fail(DIES_ECUDA, "tracker does not fit on an SM");
        const FlyPlan fp = plan_fly(m->K, m->nT, m->ldS, m->D.ldT, R.slots, true, true, logc);
        const int kf = fly_kernel(mode, true, logc);
        ge = grant_smem(kf, fp.total);
        if (ge == cudaSuccess) launch_fly(kf, grid, fp.total, 0, m->D, R, tp, fp);
    }
    if (ge != cudaSuccess) return fail(DIES_ECUDA, "trace: %s", cudaGetErrorString(ge));
    m->launches += 1;
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(events, d_ev, (size_t)count * max_events * 16, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(n_events, d_n, (size_t)count * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(DIES_ECUDA, "trace: %s", cudaGetErrorString(e));
    return DIES_OK;
}

extern "C" int dies_test_philox(uint64_t seed, uint64_t first_id, uint32_t block, uint32_t model_index, int n,
                                uint32_t* words, float* uniforms)
{
    if (!words || !uniforms || n < 1) return fail(DIES_EINVAL, "bad arguments");
    int rc = check_device();
    if (rc) return rc;
    uint32_t* dw = nullptr; float* du = nullptr;
    CUDA_TRY(cudaMalloc(&dw, (size_t)n * 16));
    if (cudaMalloc(&du, (size_t)n * 16) != cudaSuccess) { cudaFree(dw); return fail(DIES_ECUDA, "cudaMalloc failed"); }
    k_test_philox<<<(n + 255) / 256, 256>>>((uint32_t)seed, (uint32_t)(seed >> 32), first_id, block, model_index, n, dw, du);
    cudaError_t e = cudaMemcpy(words, dw, (size_t)n * 16, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(uniforms, du, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(dw); cudaFree(du);
    if (e != cudaSuccess) return fail(DIES_ECUDA, "philox test: %s", cudaGetErrorString(e));
    return DIES_OK;
}

// ------------------------------------------------------------------ atomic-unit microbenchmark (measurement support)
// The absorption step of the tracker as a stand-alone loop: every lane draws a shell (uniform over n_addr tallies,
// 8 bytes apart like the tallies of a model), the warp aggregates equal shells with __match_any_sync when asked to,
// and one lane per distinct shell issues a RETURNING 64-bit atomicAdd whose result every lane consumes.
__global__ void k_bench_atomics(unsigned long long* tallies, int n_addr, int stride, const unsigned short* __restrict__ lut,
                                int aggregate, int iters, unsigned long long* sink, unsigned long long* n_atomics)
{
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    uint32_t x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    unsigned long long acc = 0, issued = 0;
    for (int it = 0; it < iters; it++) {
        x = x * 1664525u + 1013904223u;
        // uniform over the tallies, or the workload's shell histogram through a 4096-entry look-up table
        const int j = lut ? (int)__ldg(lut + (x >> 20)) : (int)(((unsigned long long)(x >> 8) * (unsigned)n_addr) >> 24);
        unsigned long long old;
        if (aggregate) {
            const unsigned peers = __match_any_sync(0xffffffffu, j);
            const int leader = __ffs(peers) - 1;
            old = 0;
            if ((int)lane == leader) { old = atomicAdd(&tallies[(size_t)j * stride], (unsigned long long)__popc(peers)); issued++; }
            old = __shfl_sync(0xffffffffu, old, leader) + (unsigned long long)__popc(peers & lt_mask);
        } else {
            old = atomicAdd(&tallies[(size_t)j * stride], 1ull);
            issued++;
        }
        acc += old;
    }
    if (acc == 0x123456789abcdefull) *sink = acc;       // keeps the returned values alive
    for (int o = 16; o > 0; o >>= 1) issued += __shfl_xor_sync(0xffffffffu, issued, o);
    if (lane == 0) atomicAdd(n_atomics, issued);
}

extern "C" int dies_bench_atomics(int n_addr, const double* weights, int aggregate, int iters, double* lane_ops_per_s,
                                  double* atomics_per_s)
{
    const int stride = tuning().atom_stride;     // 64-bit words between two tallies
    if (n_addr < 1 || n_addr > 65535 || iters < 1 || !lane_ops_per_s || !atomics_per_s)
        return fail(DIES_EINVAL, "bad arguments");
    // look-up table of the histogram: entry e holds the tally whose cumulative weight covers (e + 0.5) / 4096
    std::vector<unsigned short> lut;
    if (weights) {
        double tot = 0.0;
        for (int i = 0; i < n_addr; i++) { if (!(weights[i] >= 0.0)) return fail(DIES_EINVAL, "negative weight"); tot += weights[i]; }
        if (!(tot > 0.0)) return fail(DIES_EINVAL, "weights sum to zero");
        lut.resize(4096);
        double c = 0.0; int i = 0;
        for (int e = 0; e < 4096; e++) {
            const double u = (e + 0.5) / 4096.0 * tot;
            while (i < n_addr - 1 && c + weights[i] <= u) c += weights[i++];
            lut[e] = (unsigned short)i;
        }
    }
    int rc = check_device();
    if (rc) return rc;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    unsigned long long* buf = nullptr;
    CUDA_TRY(cudaMalloc(&buf, ((size_t)n_addr * stride + 2) * 8 + 4096 * 2));
    unsigned short* d_lut = nullptr;
    if (weights) {
        d_lut = reinterpret_cast<unsigned short*>(buf + (size_t)n_addr * stride + 2);
        if (cudaMemcpy(d_lut, lut.data(), 4096 * 2, cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(buf); return fail(DIES_ECUDA, "copy failed"); }
    }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 4, block = 256;
    float best = 1e30f;
    unsigned long long issued = 0;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 4 && e == cudaSuccess; rep++) {          // first repetition warms up
        cudaMemset(buf, 0, ((size_t)n_addr * stride + 2) * 8);
        cudaEventRecord(e0);
        k_bench_atomics<<<grid, block>>>(buf, n_addr, stride, d_lut, aggregate, iters, buf + (size_t)n_addr * stride, buf + (size_t)n_addr * stride + 1);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
        if (e == cudaSuccess) e = cudaMemcpy(&issued, buf + (size_t)n_addr * stride + 1, 8, cudaMemcpyDeviceToHost);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return fail(DIES_ECUDA, "atomic benchmark: %s", cudaGetErrorString(e));
    *lane_ops_per_s = (double)grid * block * iters / (best * 1e-3);
    *atomics_per_s = (double)issued / (best * 1e-3);
    return DIES_OK;
}
