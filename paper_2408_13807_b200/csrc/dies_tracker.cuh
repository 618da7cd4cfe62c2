// dies_tracker.cuh -- the persistent-thread IRE package tracker for sm_100a (hot path of include/dies.h).
//
// One photon package per lane.  A warp alternates between
//   (1) an EVENT phase (all 32 lanes converged): escapes are tallied, free lanes are refilled from the model's
//       global package counter, absorptions update the 64-bit fixed-point shell tallies (one returning atomic
//       per distinct shell in the warp), then every lane that launches / scatters / re-emits runs ONE shared
//       instruction stream (event_step): a Philox4x32-10 block, two new free paths (Eq. 1), a table
//       search for the new frequency (launch and re-emission share it), the new direction, and the set-up of
//       the next flight;
//   (2) a CROSSING phase: the shell-crossing loop (Eq. 4) with no random numbers, no global
//       memory and no branches (every crossing is predicated on the lane still flying), run until fewer than a
//       set fraction of the warp's packages are still flying.
// Differences from the paper's OpenCL design are listed in DESIGN.md ("What differs from the paper").
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dies {

constexpr int kBlock = 256;          // threads per block
constexpr int kMinBlocks = 3;        // resident blocks per SM asked from the compiler
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kChunk = 128;     // package ids a warp takes from the global counter at a time
constexpr int kUnroll = 4;           // crossings per vote in the crossing loop

// event counters (same order as DIES_C_* in include/dies.h): the frequent ones are kept in registers, the rare
// ones go through shared-memory atomics
enum { LC_PACKAGES = 0, LC_CROSSINGS, LC_FFI_CROSSINGS, LC_SCATTERINGS, LC_ABSORPTIONS, LC_ESCAPED, LC_UNINTERACTED,
       LC_TERMINATED, LC_EXTRA_BLOCKS, LC_CLAMP_HI, LC_INJECTED_RAW, LC_N };

struct ModelParams {
    int Np;            // internal shells = n_shells + cav
    int cav;           // 1 if r_bounds[0] > 0: internal shell 0 is the empty cavity (R10)
    int has_ext, has_point;
    float r0hat;       // r_bounds[0] / R
    float qs_ext, qs_point;   // e_src / e_ref (<= 1): raw units per unit-weight package / 2^S
    float colmax;      // a column (units of 1/kappa_ref) larger than that of any chord: start of a dry FFI flight
};

// The shell table of one model is "unfolded" along a chord: entry c in [-ldS, ldS+1] (stored at c + ldS)
// describes the surface passage a package makes when it reaches boundary |c| moving inward (c <= 0) or outward
// (c > 0):  .x = (r_|c| / R)^2,  .y = rho^ of the shell it traverses on the way to that surface (shell |c| for
// c <= 0, shell c-1 for c > 0) with the SIGN BIT SET for inward entries.  A flight walks the table upwards; an
// inward surface that the chord does not reach (r^2 < b^2) sends it to the mirrored entry 1 - c.  Entry Np + 1
// is a sentinel with a negative r^2: a package that has left the model stops there.
struct DeviceModel {
    int N, K, nT, n_models;
    int ldS;                         // leading dimension of the per-model shell arrays (N + 1)
    int ldT;                         // entries of the unfolded shell table per model (2 ldS + 2)
    const float4* bintab;            // K: {1/kappa_abs^, 1/kappa_sca^, g, kappa_ext^}  (kappa^ = kappa / kappa_ref)
    const float* omega;              // K: albedo
    const float* epsgrid;            // nT: eps_t / eps_ref
    const float* F;                  // nT x K row CDFs of the re-emission spectra
    const float2* stab;              // n_models x ldT unfolded shell table
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

__device__ __forceinline__ float sqrt_ftz(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// one entry of the unfolded shell table from its shared-memory address (the table is read-only while packages fly)
__device__ __forceinline__ float2 lds_entry(unsigned a)
{
    float2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}

// smallest k in [0, n) with cdf[k] > u (= #{i < n-1 : cdf[i] <= u} for a non-decreasing cdf with cdf[n-1] > u):
// binary lifting with a warp-uniform trip count (top = largest power of two <= n-1, 0 if n == 1)
__device__ __forceinline__ int sample_cdf(const float* __restrict__ cdf, int n, int top, float u)
{
    int k = 0;
    for (int step = top; step > 0; step >>= 1) {
        const int t = k + step;
        if (t < n && __ldg(cdf + t - 1) <= u) k = t;
    }
    return k;
}

// t(eps) = #{j : grid[j] <= eps} clamped to n-1, given a lower bound t0 <= t(eps): the table row of a cell
// emitting eps (R4).  Rows only move up during a run, so the scan from the block's last known row is short.
__device__ __forceinline__ int row_from(const float* grid, int n, int t0, float eps)
{
    int t = t0;
    if (grid[min(t + 8, n - 1)] <= eps) {          // far away (first touch of a shell): bisect (t+8, n]
        int lo = min(t + 8, n - 1) + 1, hi = n;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (grid[mid] > eps) hi = mid; else lo = mid + 1;
        }
        return min(lo, n - 1);
    }
    while (t < n - 1 && grid[t] <= eps) t++;
    return t;
}

// Henyey-Greenstein deflection cosine (Eq. 6), inverse CDF; |g| < 1e-3 is isotropic
__device__ __forceinline__ float hg_cos(float g, float u)
{
    if (fabsf(g) < 1e-3f) return 2.f * u - 1.f;
    const float t = (1.f - g * g) / (1.f - g + 2.f * g * u);
    return (1.f + g * g - t * t) / (2.f * g);
}

// 64-bit shared-memory tally as two 32-bit words (native ATOMS.ADD instead of a 64-bit CAS loop)
__device__ __forceinline__ void smem_add64(unsigned* lo, unsigned* hi, unsigned long long v)
{
    const unsigned vlo = (unsigned)v, vhi = (unsigned)(v >> 32);
    const unsigned old = atomicAdd(lo, vlo);
    const unsigned up = vhi + ((old + vlo < old) ? 1u : 0u);
    if (up) atomicAdd(hi, up);
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
__global__ void __launch_bounds__(kBlock, kMinBlocks) dies_track(DeviceModel D, RunParams R, TraceParams tp)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = D.K, nT = D.nT, ldS = D.ldS, ldT = D.ldT;
    // shared-memory layout
    float4* s_bin = reinterpret_cast<float4*>(smem_raw);                          // K
    double* s_cs = reinterpret_cast<double*>(s_bin + K);                          // ldS
    float2* s_tab = reinterpret_cast<float2*>(s_cs + ldS);                        // ldT unfolded shell table
    float* s_eps = reinterpret_cast<float*>(s_tab + ldT);                         // nT
    float* s_omega = s_eps + nT;                                                  // K
    int* s_row = reinterpret_cast<int*>(s_omega + K);                             // ldS: fixed rows / row hints
    unsigned* s_esc = reinterpret_cast<unsigned*>(s_row + ldS);                   // 2K: low words, high words
    unsigned* s_A = s_esc + 2 * K;                                                // 2 ldS (MODE 1)
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_cnt[LC_N];      // rare counters, flushed at kernel end

    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    int top = 0;                                     // largest power of two <= K-1 (trip count of sample_cdf)
    for (int t = 1; t <= K - 1; t <<= 1) top = t;

    for (int x = tid; x < K; x += kBlock) { s_bin[x] = D.bintab[x]; s_omega[x] = D.omega[x]; }
    for (int x = tid; x < nT; x += kBlock) s_eps[x] = D.epsgrid[x];

    if (tid < LC_N) s_cnt[tid] = 0ull;
    // warp-uniform counters (identical in all lanes) and per-lane sums
    unsigned long long wc_pkg = 0, wc_sca = 0, wc_abs = 0, wc_esc = 0;
    unsigned long long lc_cross = 0, lc_ffi = 0, inj_raw = 0;

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
        for (int x = tid; x < ldT; x += kBlock) s_tab[x] = D.stab[(size_t)m * ldT + x];
        for (int x = tid; x < ldS; x += kBlock) {
            s_cs[x] = D.cscale[(size_t)m * ldS + x];
            s_row[x] = (MODE == 1) ? D.fixed_row[(size_t)m * ldS + x] : 0;
            s_A[x] = 0u; s_A[ldS + x] = 0u;
        }
        for (int x = tid; x < 2 * K; x += kBlock) s_esc[x] = 0u;
        __syncthreads();

        unsigned long long* const gA = D.A + (size_t)m * ldS;
        unsigned long long* const g_next = D.next_id + m;
        const float* const g_src = D.srccdf + (size_t)m * 2 * K;
        const unsigned long long n_ids = R.n_run * (unsigned long long)(mp.has_ext + mp.has_point);
        const unsigned tab0 = (unsigned)__cvta_generic_to_shared(s_tab) + 8u * (unsigned)ldS;   // address of entry c = 0
        const unsigned pa_out = tab0 + 8u * (unsigned)(Np + 1);                     // the sentinel beyond the outer surface

        // ---------------- per-lane package state
        // flight: along-ray coordinate s and impact parameter^2 b2 (units of R), remaining column col (units of
        // 1/kappa_ref) to the next event, shared-memory address pa of the candidate surface passage (entry E);
        // (pa - pa0) / 8 counts the passages of this flight.  alive = still flying; a lane stops either on an unreachable surface
        // (col untouched, >= 0) or because the column ran out (the passage is committed and col < 0).
        bool has = false, alive = false, launch = false;
        float s = 0.f, b2 = 0.f, col = -1.f;
        float2 E = make_float2(0.f, 0.f);
        unsigned pa = tab0, pa0 = tab0;
        int k = 0;
        bool ev_absorb = false, dry = false;         // type of the pending event; dry FFI flight (Eq. 9)
        unsigned blk = 0, ncross = 0;
        unsigned long long id = 0, q = 0;
        int n_ev = 0, pkg = 0;
        // warp-uniform id chunk
        unsigned long long ch_next = 0, ch_end = 0;
        bool exhausted = false;
        if (TRACE) {
            pkg = blockIdx.x * kBlock + tid;
            exhausted = true;
            if (pkg < tp.count) { launch = true; id = tp.first_id + (unsigned long long)pkg; }
        }

        for (;;) {
            // ======== uniform point: all 32 lanes converged ========
            const bool stopped = has && !alive;
            const bool isev = stopped && (col < 0.f);          // the column ran out: scattering or absorption
            const bool atend = stopped && !isev;               // stopped on the sentinel: left the model
            if (stopped) {
                const unsigned n = ((pa - pa0) >> 3) - (isev ? 1u : 0u);
                if (dry) lc_ffi += n; else { lc_cross += n; ncross += n; }
            }
            // (1) escapes (PAPER.md L87 last sentence)
            const bool esc = atend && !dry;
            const bool dryend = atend && dry;
            const unsigned escmask = __ballot_sync(kFull, esc);
            if (escmask) {
                if (esc) {
                    if (!TRACE) smem_add64(&s_esc[k], &s_esc[K + k], q);
                    record<TRACE>(tp, pkg, n_ev, 3 /*ESCAPE*/, D.N - 1, k, ncross);
                    if (TRACE) tp.n_events[pkg] = n_ev;
                    has = false;
                }
                wc_esc += __popc(escmask);
            }
            // (2) refill free lanes from the global package counter
            if (!exhausted) {
                const bool need = !has;
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
                        launch = true;
                        blk = 0;
                    }
                }
            }
            if (!__ballot_sync(kFull, has || launch)) break;

            // (3) absorptions: add the package's quantum to the shell tally, keep the old value (L87)
            const bool isabs = isev && ev_absorb;
            const bool issca = isev && !ev_absorb;
            // shell of the event: the one traversed on the way to the surface entry before pa, which was not reached
            const int ci = (int)(pa - tab0) / 8 - 1;
            int j = ci <= 0 ? -ci : ci - 1;
            const unsigned absmask = __ballot_sync(kFull, isabs);
            wc_abs += __popc(absmask);
            wc_sca += __popc(__ballot_sync(kFull, issca));
            wc_pkg += __popc(__ballot_sync(kFull, launch));
            unsigned long long old = 0;
            if (absmask) {
                if (TRACE) {
                    if (isabs && MODE == 0) old = gA[j];
                } else if (MODE == 1) {
                    if (isabs) smem_add64(&s_A[j], &s_A[ldS + j], q);
                } else if (R.uniform_q) {
                    const unsigned peers = __match_any_sync(kFull, isabs ? j : -1 - lane);
                    const int leader = __ffs(peers) - 1;
                    if (isabs && lane == leader) old = atomicAdd(&gA[j], q * (unsigned long long)__popc(peers));
                    old = __shfl_sync(kFull, old, leader) + q * (unsigned long long)__popc(peers & lt_mask);
                } else if (isabs) {
                    old = atomicAdd(&gA[j], q);
                }
            }

            // (4) events: launch / scatter / absorb + re-emit / end of a dry FFI flight; one Philox block each
            //     (DESIGN.md RNG contract), one instruction stream for all of them
            if (launch || isev || dryend) {
                uint32_t xw[4];
                const bool atsrc = launch || dryend;                            // the event site is the source
                const bool point = atsrc && (mp.has_ext ? ((id - R.id_base) >= R.n_total) : true);
                const float* cdf = nullptr;          // table the new frequency bin is drawn from (launch, re-emission)
                if (isabs) {
                    int row;
                    if (MODE == 1) {
                        row = s_row[j];
                    } else {
                        // emitted power per mass before and after this absorption; rows of the table (R4)
                        const double cs = s_cs[j];
                        const float eps_old = (float)((double)old * cs);
                        const float eps_new = (float)((double)(old + q) * cs);
                        const int hint = s_row[j];
                        row = row_from(s_eps, nT, hint, eps_old);
                        if (row > hint) atomicMax(&s_row[j], row);
                        const bool same = (row == nT - 1) || (eps_new < s_eps[row]);
                        if (eps_new >= s_eps[nT - 1]) atomicAdd(&s_cnt[LC_CLAMP_HI], 1ull);
                        if (!same) {
                            philox4x32_10(R.key0, R.key1, (uint32_t)id, (uint32_t)(id >> 32), blk++, (uint32_t)m, xw);
                            const float es = eps_old + uniform24(xw[0]) * (eps_new - eps_old);
                            row = row_from(s_eps, nT, row, es);
                            atomicAdd(&s_cnt[LC_EXTRA_BLOCKS], 1ull);
                        }
                    }
                    cdf = D.F + (size_t)row * K;
                } else if (launch) {
                    cdf = g_src + (point ? K : 0);                              // L55 source spectrum table
                }
                // block 0 belongs to the launch; with FFI the end of the dry flight draws it again
                const unsigned b = dryend ? 0u : blk;
                philox4x32_10(R.key0, R.key1, (uint32_t)id, (uint32_t)(id >> 32), b, (uint32_t)m, xw);
                blk = (launch && R.ffi) ? 0u : b + 1u;
                const float u0 = uniform24(xw[0]), u1 = uniform24(xw[1]);
                const float tauS = -logf(uniform24(xw[2]));      // Eq. 1
                const float tauA = -logf(uniform24(xw[3]));
                if (cdf) k = sample_cdf(cdf, K, top, u0);        // new frequency bin (launch: L55; re-emission: L87, R4)

                // ---- event site (radius re, re2 = re^2, shell j) and new direction cosine mu w.r.t. the radius
                float re, re2, mu, b2src = 0.f;
                if (atsrc) {
                    // ---- launch
                    float w = 1.f;
                    if (!point) {
                        float mu_in;
                        if (R.k_bg == 0.5f) {
                            mu_in = sqrtf(u1);                                 // Eq. 2
                            b2src = 1.f - u1;
                        } else {
                            const float l2 = log2f(u1);                        // Eq. 5: mu = u^k_bg,
                            mu_in = exp2f(R.k_bg * l2);                        //        W = 2 k_bg mu^(2-1/k_bg)
                            w = 2.f * R.k_bg * exp2f((2.f * R.k_bg - 1.f) * l2);
                            b2src = (1.f - mu_in) * (1.f + mu_in);
                        }
                        mu = -mu_in; re = 1.f; re2 = 1.f;
                        j = Np - 1;
                    } else {
                        mu = 1.f; re = mp.r0hat; re2 = re * re; j = mp.cav;   // L65, R9: radial
                    }
                    if (launch) {
                        ncross = 0; n_ev = 0; has = true; launch = false;
                        q = (unsigned long long)__float2ll_rn(w * (point ? mp.qs_point : mp.qs_ext) * R.qscale);
                        inj_raw += q;
                        record<TRACE>(tp, pkg, n_ev, 0 /*LAUNCH*/, j - mp.cav, k, 0);
                    }
                } else {
                    // ---- the step is truncated where the column ran out (L85 / L87): the surface passage
                    //      before pa was committed with col < 0, so the site lies col / rho^ before it
                    const float se = s + col / fabsf(lds_entry(pa - 8u).y);
                    re2 = fmaf(se, se, b2);
                    re = sqrtf(re2);
                    mu = 2.f * u1 - 1.f;             // re-emission: isotropic (L87)
                    if (issca) {
                        // ---- scattering with the HG phase function (L85, L167)
                        float mu0 = re > 0.f ? se / re : 1.f;
                        mu0 = fminf(1.f, fmaxf(-1.f, mu0));
                        const float ct = hg_cos(s_bin[k].z, u0);
                        const float sm = sqrtf(fmaxf(1.f - mu0 * mu0, 0.f));
                        const float sth = sqrtf(fmaxf(1.f - ct * ct, 0.f));
                        mu = mu0 * ct + sm * sth * cospif(2.f * u1);
                        mu = fminf(1.f, fmaxf(-1.f, mu));
                    }
                    record<TRACE>(tp, pkg, n_ev, issca ? 1 /*SCATTER*/ : 2 /*ABSORB*/, j - mp.cav, k, ncross);
                }
                // ---- column (in units of 1/kappa_ref) to the next event and its type
                if (R.ffi && atsrc) {
                    if (!dryend) {
                        // forced first interaction (Eq. 9-12, R11): a dry flight along the whole chord first
                        col = mp.colmax; dry = true;
                    } else {
                        const float kext = s_bin[k].w;
                        const float tau0 = kext * (mp.colmax - col);           // Eq. 9
                        const float P = -expm1f(-tau0);                        // Eq. 12
                        const unsigned long long q_un = min(q, (unsigned long long)__float2ll_rn((float)q * expf(-tau0)));
                        if (!TRACE && q_un) smem_add64(&s_esc[k], &s_esc[K + k], q_un);   // un-interacted share escapes in bin k
                        q -= q_un;
                        dry = false;
                        if (!(tau0 > 0.f)) {
                            atomicAdd(&s_cnt[LC_UNINTERACTED], 1ull);
                            record<TRACE>(tp, pkg, n_ev, 5 /*UNINTERACTED*/, j - mp.cav, k, 0);
                            if (TRACE) tp.n_events[pkg] = n_ev;
                            has = false;
                        } else {
                            const float tauE = -log1pf(-uniform24(xw[2]) * P);  // Eq. 10
                            ev_absorb = !(uniform24(xw[3]) < s_omega[k]);
                            col = tauE / kext;
                        }
                    }
                } else {
                    // L85/L87; R7 tie -> absorption; R15 one column instead of two clocks
                    const float4 bt = s_bin[k];
                    const float cA = tauA * bt.x, cS = tauS * bt.y;
                    ev_absorb = (cA <= cS);
                    col = fminf(cA, cS);
                }
                // ---- next flight: from shell j towards its inner (s < 0) or outer surface
                s = re * mu;
                b2 = (atsrc && !point) ? b2src : re2 * (1.f - mu) * (1.f + mu);
                pa = tab0 + 8u * (unsigned)((s < 0.f) ? -j : j + 1);
                pa0 = pa;
                E = lds_entry(pa);
                alive = has;
            }
            if (!has) { alive = false; col = -1.f; }             // parked lane: never flies, never looks stopped short

            // ======== crossing phase (Eq. 4): no RNG, no global memory, no branches ========
            // One crossing: d = r_c^2 - b^2 (negative: the surface is not reached, the lane stops with col
            // untouched); along-ray coordinate of the surface sn = +-sqrt(d); col -= rho^ (sn - s) (Eq. 4) is
            // committed together with the passage, and the lane stops if col < 0: the event lies col / rho^
            // before the surface (R7: an event exactly on a surface is a passage).
            const int thr = max(1, (__popc(__ballot_sync(kFull, has)) * R.thr_num) >> 5);
            for (;;) {
#pragma unroll
                for (int u = 0; u < kUnroll; u++) {
                    const float d = E.x - b2;
                    alive = alive && (d >= 0.f);
                    if (alive) {
                        const float sn = __int_as_float(__float_as_int(sqrt_ftz(d)) | (__float_as_int(E.y) & 0x80000000));
                        col = fmaf(-fabsf(E.y), sn - s, col);
                        s = sn;
                        pa += 8u;
                        E = lds_entry(pa);
                    }
                    alive = alive && (col >= 0.f);
                }
                if (!alive && (col >= 0.f)) {
                    if (__float_as_int(E.y) < 0) {
                        // the inner surface is not reached (tangent shell): head for the outer one instead
                        // entry c -> entry 1 - c; the 1 - 2c entries skipped are no passages
                        const unsigned np = 2u * tab0 + 8u - pa;
                        pa0 += np - pa;
                        pa = np;
                        E = lds_entry(pa);
                        alive = true;
                    } else if (pa != pa_out) {
                        b2 = E.x;                                // outward, b2 > r^2 by rounding only: graze
                        alive = true;
                    }
                }
                if (__popc(__ballot_sync(kFull, alive)) < thr) break;
            }
        }

        if (TRACE) break;
        // ---------------- flush the block's privatised tallies
        __syncthreads();
        unsigned long long* const gesc = D.esc + (size_t)m * K;
        for (int x = tid; x < K; x += kBlock) {
            const unsigned long long v = (unsigned long long)s_esc[x] | ((unsigned long long)s_esc[K + x] << 32);
            if (v) atomicAdd(&gesc[x], v);
        }
        if (MODE == 1)
            for (int x = tid; x < Np; x += kBlock) {
                const unsigned long long v = (unsigned long long)s_A[x] | ((unsigned long long)s_A[ldS + x] << 32);
                if (v) atomicAdd(&gA[x], v);
            }
    }

    if (TRACE) return;
    // ---------------- counters: one atomic per warp / per block (rare ones)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        inj_raw += __shfl_xor_sync(kFull, inj_raw, o);
        lc_cross += __shfl_xor_sync(kFull, lc_cross, o);
        lc_ffi += __shfl_xor_sync(kFull, lc_ffi, o);
    }
    if (lane == 0) {
        atomicAdd(&D.counters[LC_PACKAGES], wc_pkg);
        atomicAdd(&D.counters[LC_CROSSINGS], lc_cross);
        if (lc_ffi) atomicAdd(&D.counters[LC_FFI_CROSSINGS], lc_ffi);
        atomicAdd(&D.counters[LC_SCATTERINGS], wc_sca);
        atomicAdd(&D.counters[LC_ABSORPTIONS], wc_abs);
        atomicAdd(&D.counters[LC_ESCAPED], wc_esc);
        atomicAdd(&D.counters[LC_INJECTED_RAW], inj_raw);
    }
    __syncthreads();
    if (tid < LC_N && s_cnt[tid]) atomicAdd(&D.counters[tid], s_cnt[tid]);
}

}  // namespace dies
