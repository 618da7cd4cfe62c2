// dies_tracker.cuh -- the persistent-thread IRE package tracker for sm_100a (hot path of include/dies.h).
//
// One photon package per lane.  A warp alternates between
//   (1) an EVENT phase: escapes are tallied, free lanes are refilled from the model's global package
//       counter, absorptions update the 64-bit fixed-point shell tallies (one returning atomic per
//       distinct shell in the warp), then every lane that launches / scatters / re-emits draws ONE
//       Philox4x32-10 block and two new free paths (Eq. 1);
//   (2) a CROSSING phase: the shell-crossing loop (Eq. 4) with no random numbers and no
//       global memory, run until fewer than a set fraction of the warp's packages are still flying.
// Differences from the paper's OpenCL design are listed in DESIGN.md ("What differs from the paper").
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dies {

constexpr int kBlock = 256;          // threads per block
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kChunk = 128;     // package ids a warp takes from the global counter at a time

enum { ST_NEED = 0, ST_LAUNCH = 1, ST_FLY = 2, ST_SCATTER = 3, ST_ABSORB = 4, ST_ESCAPED = 5 };

// event counters (same order as DIES_C_* in include/dies.h): the frequent ones are kept warp-uniform in
// registers (updated from ballots), the rare ones go through shared-memory atomics
enum { LC_PACKAGES = 0, LC_CROSSINGS, LC_FFI_CROSSINGS, LC_SCATTERINGS, LC_ABSORPTIONS, LC_ESCAPED, LC_UNINTERACTED,
       LC_TERMINATED, LC_EXTRA_BLOCKS, LC_CLAMP_HI, LC_INJECTED_RAW, LC_N };

struct ModelParams {
    int Np;            // internal shells = n_shells + cav
    int cav;           // 1 if r_bounds[0] > 0: internal shell 0 is the empty cavity (R10)
    int has_ext, has_point;
    float r0hat;       // r_bounds[0] / R
    float qs_ext, qs_point;   // e_src / e_ref (<= 1): raw units per unit-weight package / 2^S
    float pad;
};

struct DeviceModel {
    int N, K, nT, n_models;
    int ldS;                         // leading dimension of the per-model shell arrays (N + 1)
    const float4* bintab;            // K: {1/kappa_abs^, 1/kappa_sca^, g, kappa_ext^}  (kappa^ = kappa / kappa_ref)
    const float* omega;              // K: albedo
    const float* epsgrid;            // nT: eps_t / eps_ref
    const float* F;                  // nT x K row CDFs of the re-emission spectra
    const float2* stab;              // n_models x 2(ldS+1): [2j] = {r2_inner(j), rho^(j)}, [2j+1] = {r2_outer(j), rho^(j)}
    const double* cscale;            // n_models x ldS: eps^ per raw tally unit
    const float* srccdf;             // n_models x 2 x K: external, point
    const ModelParams* mp;           // n_models
    const int* fixed_row;            // n_models x ldS
    unsigned long long* A;           // n_models x ldS   absorbed-energy tallies (raw fixed point)
    unsigned long long* esc;         // n_models x K     escape tallies (raw fixed point)
    unsigned long long* next_id;     // n_models         run-local package counter
    unsigned long long* counters;    // DIES_N_COUNTERS
    unsigned int* ticket;            // 1
};

struct RunParams {
    unsigned long long n_run;        // packages per source in this call
    unsigned long long id_base;      // packages per source done by earlier calls (accumulate)
    unsigned long long n_total;      // packages per source over the whole run
    uint32_t key0, key1;
    float k_bg;
    int ffi;
    int uniform_q;                   // all packages carry the same raw quantum (no k_bg, no FFI, one source)
    float qscale;                    // 2^S
    int n_tickets, parts;            // tickets = n_models * parts
    int thr_num;                     // leave the crossing loop when flying lanes < live * thr_num / 32
};

struct TraceParams {
    int model;
    unsigned long long first_id;     // global package id of the first traced package
    int count;
    int32_t* events;                 // count x max_events x 4
    int max_events;
    int32_t* n_events;               // count
};

// ------------------------------------------------------------------ RNG contract (include/dies.h)
__device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ float uniform24(uint32_t x) { return (__uint2float_rn(x >> 9) + 0.5f) * 1.1920928955078125e-07f; }

__device__ __forceinline__ float fast_sqrt(float x)
{
    float y;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// smallest k in [0, n) with cdf[k] > u   (cdf[n-1] >= 1 > u)
template <bool GLOBAL>
__device__ __forceinline__ int sample_cdf(const float* __restrict__ cdf, int n, float u)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        const float c = GLOBAL ? __ldg(cdf + mid) : cdf[mid];
        if (c > u) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// t(eps) = #{j : grid[j] <= eps} clamped to n-1: the table row of a cell emitting eps (R4)
__device__ __forceinline__ int row_of_eps(const float* grid, int n, float eps)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (grid[mid] > eps) hi = mid; else lo = mid + 1;
    }
    return min(lo, n - 1);
}

// Henyey-Greenstein deflection cosine (Eq. 6), inverse CDF; |g| < 1e-3 is isotropic
__device__ __forceinline__ float hg_cos(float g, float u)
{
    if (fabsf(g) < 1e-3f) return 2.f * u - 1.f;
    const float t = (1.f - g * g) / (1.f - g + 2.f * g * u);
    return (1.f + g * g - t * t) / (2.f * g);
}

template <bool TRACE>
__device__ __forceinline__ void record(const TraceParams& tp, int pkg, int& n_ev, int type, int shell, int bin,
                                       unsigned ncross)
{
    if (!TRACE) return;
    if (n_ev < tp.max_events) {
        int4* e = reinterpret_cast<int4*>(tp.events) + (size_t)pkg * tp.max_events + n_ev;
        *e = make_int4(type, shell, bin, (int)ncross);
    }
    n_ev++;
}

// ------------------------------------------------------------------ the tracker
// MODE 0: full IRE (returning 64-bit atomics on the global shell tallies, row from eps_old/eps_new)
// MODE 1: fixed temperature (row from fixed_row; tallies privatised in shared memory)
// TRACE : replay tp.count packages of one model, one per lane, tallies read-only, events recorded
template <int MODE, bool TRACE>
__global__ void __launch_bounds__(kBlock, 3) dies_track(DeviceModel D, RunParams R, TraceParams tp)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = D.K, nT = D.nT, ldS = D.ldS;
    // shared-memory layout (all offsets multiples of 16 bytes)
    float4* s_bin = reinterpret_cast<float4*>(smem_raw);                          // K
    unsigned long long* s_esc = reinterpret_cast<unsigned long long*>(s_bin + K);  // K
    unsigned long long* s_A = s_esc + K;                                           // ldS
    double* s_cs = reinterpret_cast<double*>(s_A + ldS);                           // ldS
    float2* s_stab = reinterpret_cast<float2*>(s_cs + ldS);                        // 2(ldS+1)
    float* s_eps = reinterpret_cast<float*>(s_stab + 2 * (ldS + 1));               // nT
    float* s_omega = s_eps + nT;                                                   // K
    float* s_src = s_omega + K;                                                    // 2K
    int* s_frow = reinterpret_cast<int*>(s_src + 2 * K);                           // ldS
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_cnt[LC_N];      // rare counters, flushed at kernel end

    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;

    for (int x = tid; x < K; x += kBlock) { s_bin[x] = D.bintab[x]; s_omega[x] = D.omega[x]; }
    for (int x = tid; x < nT; x += kBlock) s_eps[x] = D.epsgrid[x];

    if (tid < LC_N) s_cnt[tid] = 0ull;
    // warp-uniform counters (identical in all lanes) and the lane's injected raw energy
    unsigned long long wc_pkg = 0, wc_cross = 0, wc_sca = 0, wc_abs = 0, wc_esc = 0, inj_raw = 0;

    for (;;) {
        // ---------------- take a ticket: (model, part)
        int m;
        if (TRACE) {
            m = tp.model;
        } else {
            __syncthreads();
            if (tid == 0) s_ticket = atomicAdd(D.ticket, 1u);
            __syncthreads();
            const unsigned t = s_ticket;
            if (t >= (unsigned)R.n_tickets) break;
            m = (int)(t / (unsigned)R.parts);
        }
        const ModelParams mp = D.mp[m];
        const int Np = mp.Np;
        for (int x = tid; x < 2 * (ldS + 1); x += kBlock) s_stab[x] = D.stab[(size_t)m * 2 * (ldS + 1) + x];
        for (int x = tid; x < ldS; x += kBlock) {
            s_cs[x] = D.cscale[(size_t)m * ldS + x];
            s_frow[x] = D.fixed_row[(size_t)m * ldS + x];
            s_A[x] = 0ull;
        }
        for (int x = tid; x < 2 * K; x += kBlock) s_src[x] = D.srccdf[(size_t)m * 2 * K + x];
        for (int x = tid; x < K; x += kBlock) s_esc[x] = 0ull;
        __syncthreads();

        unsigned long long* const gA = D.A + (size_t)m * ldS;
        unsigned long long* const g_next = D.next_id + m;
        const unsigned long long n_ids = R.n_run * (unsigned long long)(mp.has_ext + mp.has_point);

        // ---------------- per-lane package state
        int st = ST_NEED;
        float b2 = 0.f, s = 0.f, col = 0.f, r2in = 0.f, r2out = 1.f, rho = 0.f;
        int j = 0, k = 0, ev_absorb = 0;
        unsigned blk = 0, ncross = 0;
        unsigned long long id = 0, q = 0;
        int n_ev = 0, pkg = 0;
        // warp-uniform id chunk
        unsigned long long ch_next = 0, ch_end = 0;
        bool exhausted = false;
        if (TRACE) {
            pkg = blockIdx.x * kBlock + tid;
            exhausted = true;
            if (pkg < tp.count) { st = ST_LAUNCH; id = tp.first_id + (unsigned long long)pkg; }
        }

        for (;;) {
            // ======== uniform point: all 32 lanes converged ========
            // (1) escapes: warp-first reduction of the escape tally (PAPER.md L87 last sentence)
            const bool esc = (st == ST_ESCAPED);
            const unsigned escmask = __ballot_sync(kFull, esc);
            if (escmask) {
                if (!TRACE) {
                    if (R.uniform_q) {
                        const unsigned peers = __match_any_sync(kFull, esc ? k : -1 - lane);
                        if (esc && lane == __ffs(peers) - 1) atomicAdd(&s_esc[k], q * (unsigned long long)__popc(peers));
                    } else if (esc) {
                        atomicAdd(&s_esc[k], q);
                    }
                }
                if (esc) {
                    record<TRACE>(tp, pkg, n_ev, 3 /*ESCAPE*/, D.N - 1, k, ncross);
                    if (TRACE) tp.n_events[pkg] = n_ev;
                    st = ST_NEED;
                }
                wc_esc += __popc(escmask);
                wc_cross += __reduce_add_sync(kFull, esc ? ncross : 0u);
            }
            // (2) refill free lanes from the global package counter
            if (!exhausted) {
                const bool need = (st == ST_NEED);
                const unsigned needmask = __ballot_sync(kFull, need);
                if (needmask) {
                    const unsigned cnt = __popc(needmask);
                    unsigned rank = __popc(needmask & lt_mask);
                    const unsigned long long avail = ch_end - ch_next;
                    unsigned long long jdx = ch_next + rank;
                    bool got = need && (rank < avail);
                    if (avail >= cnt) {
                        ch_next += cnt;
                    } else {
                        unsigned long long base = 0;
                        if (lane == 0) base = atomicAdd(g_next, (unsigned long long)kChunk);
                        base = __shfl_sync(kFull, base, 0);
                        unsigned long long nend = base + kChunk;
                        if (nend > n_ids) nend = n_ids;
                        if (base >= n_ids) { exhausted = true; nend = base; }
                        if (need && rank >= avail) {
                            jdx = base + (rank - avail);
                            got = jdx < nend;
                        }
                        ch_next = base + (cnt - avail);
                        if (ch_next > nend) ch_next = nend;
                        ch_end = nend;
                    }
                    if (got) {
                        // run-local index -> source and global package id (R2)
                        const bool second = jdx >= R.n_run;
                        id = (second ? R.n_total + (jdx - R.n_run) : jdx) + R.id_base;
                        st = ST_LAUNCH;
                        blk = 0;
                    }
                }
            }
            const unsigned live = __ballot_sync(kFull, st != ST_NEED);
            if (!live) break;

            // (3) absorptions: add the package's quantum to the shell tally, keep the old value (L87)
            const bool isabs = (st == ST_ABSORB);
            const unsigned absmask = __ballot_sync(kFull, isabs);
            wc_abs += __popc(absmask);
            wc_sca += __popc(__ballot_sync(kFull, st == ST_SCATTER));
            wc_pkg += __popc(__ballot_sync(kFull, st == ST_LAUNCH));
            unsigned long long old = 0;
            if (absmask) {
                if (TRACE) {
                    if (isabs && MODE == 0) old = gA[j];
                } else if (MODE == 1) {
                    if (isabs) atomicAdd(&s_A[j], q);
                } else if (R.uniform_q) {
                    const unsigned peers = __match_any_sync(kFull, isabs ? j : -1 - lane);
                    const int leader = __ffs(peers) - 1;
                    if (isabs && lane == leader) old = atomicAdd(&gA[j], q * (unsigned long long)__popc(peers));
                    old = __shfl_sync(kFull, old, leader) + q * (unsigned long long)__popc(peers & lt_mask);
                } else if (isabs) {
                    old = atomicAdd(&gA[j], q);
                }
            }

            // (4) events: launch / scatter / absorb+re-emit; one Philox block each (DESIGN.md RNG contract)
            if (st == ST_LAUNCH || st == ST_SCATTER || isabs) {
                uint32_t xw[4];
                int row = 0;
                if (isabs) {
                    if (MODE == 1) {
                        row = s_frow[j];
                    } else {
                        // emitted power per mass before and after this absorption; rows of the table (R4)
                        const double cs = s_cs[j];
                        const float eps_old = (float)((double)old * cs);
                        const float eps_new = (float)((double)(old + q) * cs);
                        row = row_of_eps(s_eps, nT, eps_old);
                        const bool same = (row == nT - 1) || (eps_new < s_eps[row]);
                        if (eps_new >= s_eps[nT - 1]) atomicAdd(&s_cnt[LC_CLAMP_HI], 1ull);
                        if (!same) {
                            philox4x32_10(R.key0, R.key1, (uint32_t)id, (uint32_t)(id >> 32), blk++, (uint32_t)m, xw);
                            const float es = eps_old + uniform24(xw[0]) * (eps_new - eps_old);
                            row = row_of_eps(s_eps, nT, es);
                            atomicAdd(&s_cnt[LC_EXTRA_BLOCKS], 1ull);
                        }
                    }
                }
                philox4x32_10(R.key0, R.key1, (uint32_t)id, (uint32_t)(id >> 32), blk++, (uint32_t)m, xw);
                const float u0 = uniform24(xw[0]), u1 = uniform24(xw[1]);
                float tauS = -logf(uniform24(xw[2]));       // Eq. 1
                float tauA = -logf(uniform24(xw[3]));
                bool forced = false;

                if (st == ST_LAUNCH) {
                    // ---- launch
                    ncross = 0; n_ev = 0;
                    const bool point = mp.has_ext ? ((id - R.id_base) >= R.n_total) : true;
                    k = sample_cdf<false>(s_src + (point ? K : 0), K, u0);      // L55 source spectrum table
                    float w = 1.f;
                    if (!point) {
                        float mu_in;
                        if (R.k_bg == 0.5f) {
                            mu_in = sqrtf(u1);                                 // Eq. 2
                            b2 = 1.f - u1;
                        } else {
                            mu_in = powf(u1, R.k_bg);                          // Eq. 5
                            w = 2.f * R.k_bg * powf(u1, 2.f * R.k_bg - 1.f);
                            b2 = (1.f - mu_in) * (1.f + mu_in);
                        }
                        s = -mu_in;
                        j = Np - 1;
                    } else {
                        b2 = 0.f; s = mp.r0hat; j = mp.cav;                    // L65, R9: radial
                    }
                    const float2 pi = s_stab[2 * j], po = s_stab[2 * j + 1];
                    r2in = pi.x; r2out = po.x; rho = pi.y;
                    q = (unsigned long long)__float2ll_rn(w * (point ? mp.qs_point : mp.qs_ext) * R.qscale);
                    inj_raw += q;
                    record<TRACE>(tp, pkg, n_ev, 0 /*LAUNCH*/, j - mp.cav, k, 0);
                    if (R.ffi) {
                        // ---- forced first interaction (Eq. 9-12, R11): optical depth of the whole chord
                        float ws = s, wri = r2in, wro = r2out, wrho = rho, colsum = 0.f;
                        int wj = j;
                        unsigned wc = 0;
                        for (;;) {
                            const bool inward = (ws < 0.f) && (b2 < wri);
                            const float root = fast_sqrt(fmaxf((inward ? wri : wro) - b2, 0.f));
                            const float sn = inward ? -root : root;
                            colsum += wrho * (sn - ws);
                            ws = sn; wc++;
                            wj += inward ? -1 : 1;
                            if (wj == Np) break;
                            const float2 p = s_stab[2 * wj + (inward ? 0 : 1)];
                            if (inward) { wro = wri; wri = p.x; } else { wri = wro; wro = p.x; }
                            wrho = p.y;
                        }
                        atomicAdd(&s_cnt[LC_FFI_CROSSINGS], (unsigned long long)wc);
                        const float kext = s_bin[k].w;
                        const float tau0 = kext * colsum;
                        const float P = -expm1f(-tau0);                        // Eq. 12
                        const unsigned long long q_un = min(q, (unsigned long long)__float2ll_rn((float)q * expf(-tau0)));
                        if (!TRACE && q_un) atomicAdd(&s_esc[k], q_un);        // un-interacted share escapes in bin k
                        q -= q_un;
                        if (!(tau0 > 0.f)) {
                            atomicAdd(&s_cnt[LC_UNINTERACTED], 1ull);
                            record<TRACE>(tp, pkg, n_ev, 5 /*UNINTERACTED*/, j - mp.cav, k, 0);
                            if (TRACE) tp.n_events[pkg] = n_ev;
                            st = ST_NEED;
                        } else {
                            const float tauE = -log1pf(-uniform24(xw[2]) * P);  // Eq. 10
                            ev_absorb = !(uniform24(xw[3]) < s_omega[k]);
                            col = tauE / kext;
                            forced = true;
                        }
                    }
                } else {
                    // ---- truncate the step at the event position (L85 / L87)
                    const float se = s + col / rho;
                    const float re2 = fmaf(se, se, b2);
                    const float re = sqrtf(re2);
                    float mu;
                    if (st == ST_SCATTER) {
                        // ---- scattering with the HG phase function (L85, L167)
                        float mu0 = re > 0.f ? se / re : 1.f;
                        mu0 = fminf(1.f, fmaxf(-1.f, mu0));
                        const float ct = hg_cos(s_bin[k].z, u0);
                        const float sm = sqrtf(fmaxf(1.f - mu0 * mu0, 0.f));
                        const float sth = sqrtf(fmaxf(1.f - ct * ct, 0.f));
                        mu = mu0 * ct + sm * sth * cospif(2.f * u1);
                        mu = fminf(1.f, fmaxf(-1.f, mu));
                        record<TRACE>(tp, pkg, n_ev, 1 /*SCATTER*/, j - mp.cav, k, ncross);
                    } else {
                        // ---- absorption + immediate re-emission (L87): new frequency from the row CDF,
                        //      isotropic direction, same position, same energy
                        k = sample_cdf<true>(D.F + (size_t)row * K, K, u0);
                        mu = 2.f * u1 - 1.f;
                        record<TRACE>(tp, pkg, n_ev, 2 /*ABSORB*/, j - mp.cav, k, ncross);
                    }
                    s = re * mu;
                    b2 = re2 * (1.f - mu) * (1.f + mu);
                }
                if (st != ST_NEED) {
                    if (!forced) {
                        // column (in units of 1/kappa_ref) to the next event and its type (L85/L87; R7 tie -> absorption)
                        const float4 bt = s_bin[k];
                        const float cA = tauA * bt.x, cS = tauS * bt.y;
                        ev_absorb = (cA <= cS);
                        col = fminf(cA, cS);
                    }
                    st = ST_FLY;
                }
            }

            // ======== crossing phase (Eq. 4): no RNG, no global memory ========
            const int thr = max(1, (__popc(live) * R.thr_num) >> 5);
            for (;;) {
                if (st == ST_FLY) {
                    const bool inward = (s < 0.f) && (b2 < r2in);
                    const float root = fast_sqrt(fmaxf((inward ? r2in : r2out) - b2, 0.f));
                    const float sn = inward ? -root : root;
                    const float dcol = rho * (sn - s);
                    if (col < dcol) {
                        st = ev_absorb ? ST_ABSORB : ST_SCATTER;
                    } else {
                        col -= dcol;
                        s = sn;
                        ncross++;
                        j += inward ? -1 : 1;
                        const float2 p = s_stab[2 * j + (inward ? 0 : 1)];
                        if (inward) { r2out = r2in; r2in = p.x; } else { r2in = r2out; r2out = p.x; }
                        rho = p.y;
                        if (j == Np) st = ST_ESCAPED;
                    }
                }
                const unsigned fl = __ballot_sync(kFull, st == ST_FLY);
                if (__popc(fl) < thr) break;
            }
        }

        if (TRACE) break;
        // ---------------- flush the block's privatised tallies
        __syncthreads();
        unsigned long long* const gesc = D.esc + (size_t)m * K;
        for (int x = tid; x < K; x += kBlock) { const unsigned long long v = s_esc[x]; if (v) atomicAdd(&gesc[x], v); }
        if (MODE == 1)
            for (int x = tid; x < Np; x += kBlock) { const unsigned long long v = s_A[x]; if (v) atomicAdd(&gA[x], v); }
    }

    if (TRACE) return;
    // ---------------- counters: one atomic per warp (uniform ones) / per block (rare ones)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) inj_raw += __shfl_xor_sync(kFull, inj_raw, o);
    if (lane == 0) {
        atomicAdd(&D.counters[LC_PACKAGES], wc_pkg);
        atomicAdd(&D.counters[LC_CROSSINGS], wc_cross);
        atomicAdd(&D.counters[LC_SCATTERINGS], wc_sca);
        atomicAdd(&D.counters[LC_ABSORPTIONS], wc_abs);
        atomicAdd(&D.counters[LC_ESCAPED], wc_esc);
        atomicAdd(&D.counters[LC_INJECTED_RAW], inj_raw);
    }
    __syncthreads();
    if (tid < LC_N && s_cnt[tid]) atomicAdd(&D.counters[tid], s_cnt[tid]);
}

}  // namespace dies
