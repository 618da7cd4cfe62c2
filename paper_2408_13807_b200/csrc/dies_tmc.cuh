// dies_tmc.cuh -- one iteration of the traditional Monte Carlo (TMC) with continuous absorption, the second workload
// of the tracker (R22).
//
// Every active source and the dust (each cell emitting the power per mass eps_i it absorbed in the run before) send
// n packages.  A package is followed by ONE lane from launch to escape: per crossing the unfolded shell table gives
// the column of the step (the arithmetic of the crossing step of dies_fly.cuh), the package leaves
// W (1 - e^{-kappa_A rho l}) of its energy in the cell (L37: "updates made to every cell along the photon path") and
// keeps the rest; scatterings are discrete events at tau_S = -ln u (Eq. 1).  Energies are 64-bit fixed-point
// integers as in the IRE trackers (R13): a package starts with its quantum and hands it out in integer pieces, so
// injected = absorbed + escaped + terminated holds exactly.  The pieces are cut with a carried remainder that starts
// at a uniform random offset per package (a spare word of its launch block): the deposit of a step is
// floor(acc + q f) with acc the fraction left over by the steps before, so the expectation of every deposit is the
// exact q f however small it is (thin cells, weak sources, attenuated packages: rounding each step to the nearest
// integer would leave nothing there and bias T low).  The launch quantum of a package is cut the same way.  The tallies of a block are privatised in shared memory.
// Lanes that finished their package wait until a quarter of the warp is idle, then the idle lanes launch new packages
// together; lanes whose step ended in a scattering wait for the end of the round of kTmcSteps steps and scatter together.
#pragma once
#include "dies_tracker.cuh"

namespace dies {

#ifndef DIES_TMC_STEPS
#define DIES_TMC_STEPS 12
#endif
#ifndef DIES_TMC_REFILL
#define DIES_TMC_REFILL 8
#endif
constexpr int kTmcSteps = DIES_TMC_STEPS;    // crossings between two looks at the idle lanes and the pending scatterings
constexpr int kTmcRefill = DIES_TMC_REFILL;  // idle lanes that trigger a refill

struct TmcModel {
    const float* G;                   // nT x K: row CDFs of the emission spectra themselves (thermal spectrum of T_t)
    const float* cellcdf;             // n_models x ldS: cumulative luminosity of the cells (dust packages start there)
    const int* row;                   // n_models x ldS: t_i = #{rows with eps_t <= eps_i} in [0, nT]
    const float* mix;                 // n_models x ldS: eps_{t-1} / eps_i: share of the spectrum of row t-1 (0 for t = 0,
                                      // 1 beyond the table: its last row)
    const float* qs_dust;             // n_models: dust package energy / reference energy (0: cold dust, no packages)
};

struct TmcPlan { unsigned bin, tab, cell, row, mix, esc, A, total; };
__host__ __device__ inline TmcPlan plan_tmc(int K, int ldS, int ldT)
{
    TmcPlan p;
    unsigned o = 0;
    p.bin = o;  o += 16u * K;
    p.tab = o;  o += 8u * (unsigned)(ldT + 2);
    p.cell = o; o += 4u * ldS;
    p.row = o;  o += 4u * ldS;
    p.mix = o;  o += 4u * ldS;
    p.esc = o;  o += 8u * K;
    p.A = o;    o += 8u * ldS;
    p.total = (o + 15u) & ~15u;
    return p;
}

// smallest k with cdf[k] > u by bisection (tables without a guide table; shared or global memory)
__device__ __forceinline__ int bisect_cdf(const float* cdf, int n, float u)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (cdf[mid] > u) hi = mid; else lo = mid + 1;
    }
    return lo;
}

__global__ void __launch_bounds__(kBlock, kMinBlocks) dies_tmc(DeviceModel D, RunParams R, TmcModel Tm, TmcPlan sp)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = D.K, nT = D.nT, ldS = D.ldS, ldT = D.ldT;
    float4* const s_bin = reinterpret_cast<float4*>(smem_raw + sp.bin);
    float2* const s_tab = reinterpret_cast<float2*>(smem_raw + sp.tab);
    float* const s_cell = reinterpret_cast<float*>(smem_raw + sp.cell);
    int* const s_row = reinterpret_cast<int*>(smem_raw + sp.row);
    float* const s_mix = reinterpret_cast<float*>(smem_raw + sp.mix);
    unsigned* const s_esc = reinterpret_cast<unsigned*>(smem_raw + sp.esc);
    unsigned* const s_A = reinterpret_cast<unsigned*>(smem_raw + sp.A);
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_cnt[LC_N];

    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int x = tid; x < K; x += kBlock) s_bin[x] = D.bintab[x];
    if (tid < LC_N) s_cnt[tid] = 0ull;
    unsigned lc_cross = 0, lc_sca = 0, lc_pkg = 0, lc_esc = 0, lc_term = 0;
    unsigned long long lc_inj = 0, lc_termraw = 0;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_ticket = atomicAdd(D.ticket, 1u);
        __syncthreads();
        const unsigned tk = s_ticket;
        if (tk >= (unsigned)R.n_tickets) break;
        const int m = (int)(tk / (unsigned)R.parts);
        const ModelParams mp = D.mp[m];
        const int Np = mp.Np;
        const float qs_dust = Tm.qs_dust[m];
        for (int x = tid; x < ldT; x += kBlock) s_tab[x] = D.stab[(size_t)m * ldT + x];
        for (int x = tid; x < ldS; x += kBlock) {
            s_cell[x] = Tm.cellcdf[(size_t)m * ldS + x];
            s_row[x] = Tm.row[(size_t)m * ldS + x];
            s_mix[x] = Tm.mix[(size_t)m * ldS + x];
            s_A[x] = 0u; s_A[ldS + x] = 0u;
        }
        for (int x = tid; x < 2 * K; x += kBlock) s_esc[x] = 0u;
        __syncthreads();

        unsigned long long* const g_next = D.next_id + m;
        const float* const g_src = D.srccdf + (size_t)m * 2 * K;
        const unsigned short* const g_srcguide = D.guideS + (size_t)m * 2 * kGuide;
        const int n_src = mp.has_ext + mp.has_point;
        const unsigned long long n_ids = R.n_run * (unsigned long long)(n_src + (qs_dust > 0.f ? 1 : 0));
        const unsigned tab0 = (unsigned)__cvta_generic_to_shared(s_tab) + 8u * (unsigned)ldS;
        const unsigned pa_out = tab0 + 8u * (unsigned)(Np + 1);

        // per-lane package: id, bin k, opacities of the bin, coordinate a along the entry ahead, impact parameter^2,
        // table position, remaining scattering depth, remaining quantum, relative weight, Philox block
        bool active = false, pend = false;
        unsigned long long id = 0;
        int k = 0;
        float kapA = 0.f, kapS = 0.f, g = 0.f, a = 0.f, b2 = 0.f, tauS = 0.f, w = 0.f, acc = 0.f;
        unsigned pa = tab0, qrem = 0, blk = 0;
        unsigned long long ch_next = 0, ch_end = 0;
        bool exhausted = false;

        for (;;) {
            // ---- idle lanes launch new packages together
            const unsigned idle = __ballot_sync(kFull, !active);
            if (!exhausted && (__popc(idle) >= kTmcRefill || idle == kFull)) {
                bool need = !active;
                const unsigned cntn = __popc(idle);
                const unsigned rank = __popc(idle & lt_mask);
                const unsigned long long avail = ch_end - ch_next;
                unsigned long long jdx = ch_next + rank;
                bool got = need && (rank < avail);
                if (avail >= cntn) {
                    ch_next += cntn;
                } else {
                    unsigned long long base = 0;
                    if (lane == 0) base = atomicAdd(g_next, (unsigned long long)R.chunk);
                    base = __shfl_sync(kFull, base, 0);
                    unsigned long long nend = base + R.chunk;
                    if (nend > n_ids) nend = n_ids;
                    if (base >= n_ids) { exhausted = true; nend = base; }
                    if (need && rank >= avail) { jdx = base + (rank - avail); got = jdx < nend; }
                    ch_next = base + (cntn - avail);
                    if (ch_next > nend) ch_next = nend;
                    ch_end = nend;
                }
                if (got) {
                    // run-local index -> source (external field, point source, dust) and global package id
                    const int which = (int)(jdx / R.n_run);
                    id = (unsigned long long)which * R.n_total + (jdx - (unsigned long long)which * R.n_run) + R.id_base;
                    uint32_t xw[4];
                    philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), 0u, (uint32_t)m + R.model0, xw);
                    blk = 1u;
                    float re, re2, mu, qs, uq;
                    int j;
                    if (which < n_src) {
                        // ---- a package of a source, as in the IRE method
                        const bool point = mp.has_ext ? which == 1 : true;
                        k = sample_cdf(g_src + (point ? K : 0), g_srcguide + (point ? kGuide : 0), uniform24(xw[0]));
                        if (!point) {
                            const float u1 = uniform24(xw[1]);
                            mu = -sqrtf(u1); re = 1.f; re2 = 1.f; j = Np - 1;            // Eq. 2
                        } else {
                            mu = 1.f; re = mp.r0hat; re2 = re * re; j = mp.cav;          // L65, R9
                        }
                        tauS = neg_log(uniform24(xw[2]));
                        // the spare word of the block, halved: offsets of the quantum and of the deposits
                        uq = ((float)(xw[3] >> 16) + 0.5f) * (1.f / 65536.f);
                        acc = ((float)(xw[3] & 0xffffu) + 0.5f) * (1.f / 65536.f);
                        qs = point ? mp.qs_point : mp.qs_ext;
                    } else {
                        // ---- a dust package: cell by luminosity, radius uniform in its volume (L251), isotropic,
                        //      bin from the cell's spectrum C(eps) (R22)
                        j = bisect_cdf(s_cell, Np, uniform24(xw[0]));
                        const float ri2 = s_tab[ldS - j].x, ro2 = s_tab[ldS + j + 1].x;   // entries -j and j + 1
                        const float ri = sqrtf(ri2), ro = sqrtf(ro2);
                        const float ri3 = ri * ri2, ro3 = ro * ro2;
                        re = cbrtf(fmaf(uniform24(xw[1]), ro3 - ri3, ri3));
                        re = fminf(ro, fmaxf(ri, re));
                        re2 = re * re;
                        mu = 2.f * uniform24(xw[2]) - 1.f;
                        const int t = s_row[j];
                        const bool lower = uniform24(xw[3]) < s_mix[j];
                        uint32_t xv[4];
                        philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), 1u, (uint32_t)m + R.model0, xv);
                        blk = 2u;
                        const float u0 = uniform24(xv[0]);
                        if (lower) k = bisect_cdf(Tm.G + (size_t)(t >= nT ? nT - 1 : t - 1) * K, K, u0);
                        else k = sample_cdf(D.F + (size_t)t * K, D.guideF + (size_t)t * kGuide, u0);
                        tauS = neg_log(uniform24(xv[1]));
                        uq = uniform24(xv[2]);                                           // spare words: offsets of the
                        acc = uniform24(xv[3]);                                          // quantum and of the deposits
                        qs = qs_dust;
                    }
                    const float4 bt = s_bin[k];
                    kapA = bt.x < 3.0e38f ? 1.f / bt.x : 0.f;
                    kapS = bt.y < 3.0e38f ? 1.f / bt.y : 0.f;
                    g = bt.z;
                    // quantum of the package: floor(qs 2^S + offset), so that a weak source (qs << 1, a quantum of tens
                    // or thousands of units) injects its luminosity without the bias of one fixed rounding; the
                    // reference source (qs = 1) keeps exactly 2^S
                    qrem = __float2uint_rz(fmaf(qs, R.qscale, uq));
                    w = 1.f;
                    lc_inj += qrem;
                    lc_pkg++;
                    const float s = re * mu;
                    b2 = fminf(re2 * (1.f - mu) * (1.f + mu), s_tab[ldS + j + 1].x);
                    pa = tab0 + 8u * (unsigned)((s < 0.f) ? -j : j + 1);
                    a = fabsf(s);
                    active = true;
                }
            }
            if (!__any_sync(kFull, active)) break;

            // L119: a package ends below 1e-10 of its launch weight
            auto guard = [&]() {
                if (w < 1e-10f) {
                    if (mp.cav && pa == tab0) lc_cross++;        // (ended on the wall of the cavity: R10 counts its passage whole)
                    lc_termraw += qrem;
                    lc_term++;
                    active = false;
                }
            };

            // ---- kTmcSteps crossings of every active lane.  A lane whose step ends in a scattering waits (pend) for
            //      the end of the round: the scattering code then runs once for all such lanes of the warp together
            //      instead of inside the step loop at two or three active lanes.
#pragma unroll 1
            for (int u = 0; u < kTmcSteps; u++) {
                if (!active || pend) continue;
                const float2 T = lds_entry(pa);
                const float d = T.x - b2;
                if (d < 0.f) {
                    // tangent shell: turn around (an outward surface is always reached: b2 is clamped at every launch)
                    pa = 2u * tab0 + 8u - pa; a = -a;
                    continue;
                }
                const float an = sqrt_ftz(d);
                const float dc = T.y * (an - a);                 // column of the step (>= 0), units of 1 / kappa_ref
                const float dtauS = kapS * dc;
                const bool event = tauS < dtauS;
                const float f = event ? tauS / dtauS : 1.f;
                // L37: continuous absorption along the step
                const float dtA = kapA * dc * f;
                const float frac = -expm1f(-dtA);
                // integer piece with the carried remainder (unbiased for pieces far below one unit, see the header)
                const float x = fmaf((float)qrem, frac, acc);
                const unsigned dq = min(qrem, __float2uint_rz(x));
                acc = x - (float)dq;
                const int c = (int)(pa - tab0) / 8;
                const int j = c <= 0 ? -c : c - 1;
                if (dq) smem_add64(&s_A[j], &s_A[ldS + j], (unsigned long long)dq);
                qrem -= dq;
                w *= expf(-dtA);                                 // (not 1 - frac: that cancels when little is left)
                if (event) {
                    // scattering (L85): the step is truncated at the event; the new direction follows after the round
                    a = fmaf(f, an - a, a);
                    pend = true;
                    continue;
                }
                tauS -= dtauS;
                a = an;
                pa += 8u;
                lc_cross++;
                if (pa == pa_out) {
                    // the outer surface: the package leaves the model (L87 last sentence)
                    if (qrem) smem_add64(&s_esc[k], &s_esc[K + k], (unsigned long long)qrem);
                    lc_esc++;
                    active = false;
                    continue;
                }
                guard();
            }
            if (pend) {
                // ---- scattering (L85): new direction from the HG function of the bin, at the truncated position
                const int c = (int)(pa - tab0) / 8;
                const int j = c <= 0 ? -c : c - 1;
                const float se = (pa <= tab0) ? -a : a;
                const float re2 = fmaf(se, se, b2);
                const float re = sqrtf(re2);
                float mu0 = re > 0.f ? se / re : 1.f;
                mu0 = fminf(1.f, fmaxf(-1.f, mu0));
                uint32_t xw[4];
                philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), blk++, (uint32_t)m + R.model0, xw);
                const float ct = hg_cos(g, uniform24(xw[0]));
                const float sm = sqrtf(fmaxf(1.f - mu0 * mu0, 0.f)), sth = sqrtf(fmaxf(1.f - ct * ct, 0.f));
                float mu = mu0 * ct + sm * sth * cospif(2.f * uniform24(xw[1]));
                mu = fminf(1.f, fmaxf(-1.f, mu));
                tauS = neg_log(uniform24(xw[2]));
                const float s = re * mu;
                b2 = fminf(re2 * (1.f - mu) * (1.f + mu), lds_entry(tab0 + 8u * (unsigned)(j + 1)).x);
                pa = tab0 + 8u * (unsigned)((s < 0.f) ? -j : j + 1);
                a = fabsf(s);
                lc_sca++;
                pend = false;
                guard();
            }
        }
        // ---- flush the block's privatised tallies
        __syncthreads();
        unsigned long long* const gA = D.A + (size_t)m * ldS * kTallyStride;
        unsigned long long* const gesc = D.esc + (size_t)m * K;
        for (int x = tid; x < K; x += kBlock) {
            const unsigned long long v = (unsigned long long)s_esc[x] | ((unsigned long long)s_esc[K + x] << 32);
            if (v) atomicAdd(&gesc[x], v);
        }
        for (int x = tid; x < Np; x += kBlock) {
            const unsigned long long v = (unsigned long long)s_A[x] | ((unsigned long long)s_A[ldS + x] << 32);
            if (v) atomicAdd(&gA[x * kTallyStride], v);
        }
    }
    // ---- counters
    atomicAdd(&s_cnt[LC_CROSSINGS], (unsigned long long)lc_cross);
    atomicAdd(&s_cnt[LC_SCATTERINGS], (unsigned long long)lc_sca);
    atomicAdd(&s_cnt[LC_PACKAGES], (unsigned long long)lc_pkg);
    atomicAdd(&s_cnt[LC_ESCAPED], (unsigned long long)lc_esc);
    atomicAdd(&s_cnt[LC_TERMINATED], (unsigned long long)lc_term);
    atomicAdd(&s_cnt[LC_INJECTED_RAW], lc_inj);
    atomicAdd(&s_cnt[LC_TERMINATED_RAW], lc_termraw);
    __syncthreads();
    if (tid < LC_N && s_cnt[tid]) atomicAdd(&D.counters[tid], s_cnt[tid]);
}

}  // namespace dies
