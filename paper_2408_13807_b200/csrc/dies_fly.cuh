// dies_fly.cuh -- the tracker of runs whose package weights are fixed at launch (plain, k_bg, FFI; every configuration
// of BASELINE.json).
//
// Every warp keeps a pool of P photon packages in shared memory (32 bytes each) and four stacks of pool slots: packages
// ready to fly, and packages waiting for an absorption, a scattering, or a source event (escape tally + launch of the
// next package id).  The warp alternates between
//   (1) a CROSSING phase (Eq. 4): each lane flies one package in registers.  A block of kSteps
//       predicated crossing steps (no random numbers, no global memory, no branches) is followed by a short block end
//       without votes or ranks: a tangent passage turns the flight around in place; a flight that ended (event or
//       escape) is stored into its slot, which is pushed on the stack of its event type (one shared-memory atomic gives
//       the position), and a lane without a flight pops the ready stack (one more atomic).  A stopped lane never waits
//       for other lanes to stop, and any lane flies any package.
//   (2) an EVENT phase: batches of 32 slots popped from ONE stack run one of three specialised routines on the full
//       warp: absorption + re-emission (L87), scattering (L85), or escape tally + launch of the next package id
//       (L51-65, L87, L132-149); the packages go back into their slots and onto the ready stack.  Partial batches run
//       only while too few packages are ready to fly.
// Differences from the paper's OpenCL design are listed in DESIGN.md ("What differs from the paper").
#pragma once
#include "dies_tracker.cuh"

namespace dies {

constexpr int kFlyBlock = 1024;      // threads per block: ONE block per SM, so that its 32 warps share one set of tables
constexpr int kFlyWarps = kFlyBlock / 32;
constexpr int kSteps = 8;            // crossing steps per block
constexpr int kMaxSlots = 8;         // pool slots per lane: P = 32 slots <= 256 (stack entries are bytes)
// The unfolded shell table is read once per crossing step by every lane, at an address that is random from lane to
// lane: with one copy of the table an 8-byte read of a warp takes about six passes of the shared-memory data pipe
// (measured: that pipe, not instruction issue, bounded the first kernels).  The table is therefore kept in 2^LOGC
// interleaved copies, copy (lane mod 2^LOGC) for each lane: with 16 copies the 16 lanes of a half-warp read 16
// different bank pairs whatever entries they are at -- two passes, the minimum for 256 bytes.

// the stacks of a warp: stack t holds P bytes at queues + t P, its length is word t of the warp's counter quad
enum { FQ_READY = 0, FQ_ABS, FQ_SCA, FQ_SRC, FQ_N };

// shared-memory plan of a block (byte offsets), computed by the host and passed as a kernel parameter
struct FlyPlan { unsigned bin, cs, tab, eps, omega, row, esc, A, poolA, poolB, poolQ, queues, cnt, trace, total; };
__host__ __device__ inline FlyPlan plan_fly(int K, int nT, int ldS, int ldT, int M, bool trace, bool with_q, int logc)
{
    constexpr unsigned kWarps = kFlyWarps;
    FlyPlan p;
    const unsigned P = 32u * (unsigned)M;
    unsigned o = 0;
    p.bin = o;   o += 16u * K;                       // float4 K
    p.cs = o;    o += 8u * ldS;                      // double ldS
    o = (o + 15u) & ~15u;
    o = (o + 127u) & ~127u;
    p.tab = o;   o += (8u << logc) * (unsigned)(ldT + kSteps + 2);   // float2 ldT x copies (+ the look-ahead reads of a stopped lane)
    p.eps = o;   o += 4u * nT;
    p.omega = o; o += 4u * K;
    p.row = o;   o += 4u * ldS;
    p.esc = o;   o += 8u * K;                        // low words, high words
    p.A = o;     o += 8u * ldS;                      // low words, high words (fixed-T mode)
    o = (o + 15u) & ~15u;
    p.poolA = o; o += 16u * kWarps * P;              // float4 {a, b2 (sign bit: next event is an absorption), col, c}
    p.poolB = o; o += 16u * kWarps * P;              // uint4  {id lo, id hi, blk, flags}
    p.poolQ = o; if (with_q) o += 8u * kWarps * P;   // raw quantum of the package (not stored when all are equal)
    p.queues = o; o += (unsigned)FQ_N * kWarps * P;  // byte stacks of pool slots
    o = (o + 15u) & ~15u;
    p.cnt = o;   o += 16u * kWarps;                  // int4 per warp: lengths of the four stacks

    p.trace = o; if (trace) o += 12u * kWarps * P;   // pkg, n_ev, crossings so far
    p.total = (o + 15u) & ~15u;
    return p;
}

// returning 32-bit add on a shared-memory word (the stack lengths of a warp)
__device__ __forceinline__ unsigned atoms_add(unsigned a, unsigned v)
{
    unsigned old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(v) : "memory");
    return old;
}

// new free paths at an event or a launch (Eq. 1): column (units of 1/kappa_ref) to the next event and its type.
// L85/L87; R7 tie -> absorption; R15 one column instead of two clocks
__device__ __forceinline__ void draw_column(const float4 bt, float tauS, float tauA, float& col, bool& ev_absorb)
{
    const float cA_ = tauA * bt.x, cS_ = tauS * bt.y;
    ev_absorb = (cA_ <= cS_);
    col = fminf(cA_, cS_);
}

// MODE 0: full IRE (returning 64-bit atomics on the global shell tallies, row from eps_old/eps_new)
// MODE 1: fixed temperature (row from fixed_row; tallies privatised in shared memory)
// TRACE : replay tp.count packages of one model, tallies read-only, events recorded
// LOGC : log2 of the number of interleaved copies of the shell table (4, or 0 when 16 copies do not fit)
template <int MODE, bool TRACE, int LOGC>
__global__ void __launch_bounds__(kFlyBlock, 1) dies_fly(DeviceModel D, RunParams R, TraceParams tp, FlyPlan sp)
{
    constexpr int kBlock = kFlyBlock;
    constexpr unsigned ES = 8u << LOGC;              // bytes between two entries of the lane's copy of the shell table
    constexpr int ESH = 3 + LOGC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = D.K, nT = D.nT, ldS = D.ldS, ldT = D.ldT, M = R.slots, P = 32 * M;
    float4* const s_bin = reinterpret_cast<float4*>(smem_raw + sp.bin);             // K
    double* const s_cs = reinterpret_cast<double*>(smem_raw + sp.cs);               // ldS
    float2* const s_tab = reinterpret_cast<float2*>(smem_raw + sp.tab);             // ldT unfolded shell table
    float* const s_eps = reinterpret_cast<float*>(smem_raw + sp.eps);               // nT
    float* const s_omega = reinterpret_cast<float*>(smem_raw + sp.omega);           // K
    int* const s_row = reinterpret_cast<int*>(smem_raw + sp.row);                   // ldS: fixed rows / row hints
    unsigned* const s_esc = reinterpret_cast<unsigned*>(smem_raw + sp.esc);         // 2K: low words, high words
    unsigned* const s_A = reinterpret_cast<unsigned*>(smem_raw + sp.A);             // 2 ldS (MODE 1)
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_cnt[LC_N];      // counters of the block, flushed at kernel end

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem_raw);
    const unsigned aA = sbase + sp.poolA + 16u * (unsigned)(wid * P);          // float4 {a, +-b2, col, entry index c} per slot
    const unsigned aB = sbase + sp.poolB + 16u * (unsigned)(wid * P);          // uint4 {id lo, id hi, blk, flags}
    const unsigned aQ = sbase + sp.poolQ + 8u * (unsigned)(wid * P);           // raw quantum
    const unsigned qb = sbase + sp.queues + (unsigned)(wid * FQ_N * P);        // stack t at qb + t P
    const unsigned cq = sbase + sp.cnt + 16u * (unsigned)wid;                  // lengths {ready, abs, sca, src}
    int* const pT = reinterpret_cast<int*>(smem_raw + sp.trace) + wid * 3 * P;      // TRACE only

    for (int x = tid; x < K; x += kBlock) { s_bin[x] = D.bintab[x]; s_omega[x] = D.omega[x]; }
    for (int x = tid; x < nT; x += kBlock) s_eps[x] = D.epsgrid[x];
    if (tid < LC_N) s_cnt[tid] = 0ull;

    // warp-uniform event counts and per-lane crossing counts (ES per crossing) since the last flush into s_cnt
    unsigned wc_pkg = 0, wc_sca = 0, wc_abs = 0, wc_esc = 0, lc8 = 0, lc_ffi = 0;

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
        for (int x = tid; x < (ldT << LOGC); x += kBlock) s_tab[x] = D.stab[(size_t)m * ldT + (x >> LOGC)];
        for (int x = tid; x < ldS; x += kBlock) {
            s_cs[x] = D.cscale[(size_t)m * ldS + x];
            s_row[x] = (MODE == 1) ? D.fixed_row[(size_t)m * ldS + x] : 0;
            s_A[x] = 0u; s_A[ldS + x] = 0u;
        }
        for (int x = tid; x < 2 * K; x += kBlock) s_esc[x] = 0u;
        // every slot of the pool is free and waits for a package id
        for (int x = lane; x < P; x += 32) { sts_u4(aB + 16u * x, 0u, 0u, 0u, 0u); sts_u8(qb + (unsigned)(FQ_SRC * P + x), (unsigned)x); }
        if (lane == 0) sts_u4(cq, 0u, 0u, 0u, (unsigned)P);
        __syncthreads();

        unsigned long long* const gA = D.A + (size_t)m * ldS * kTallyStride;
        unsigned long long* const g_next = TRACE ? tp.counter : D.next_id + m;
        const float* const g_src = D.srccdf + (size_t)m * 2 * K;
        const unsigned short* const g_srcguide = D.guideS + (size_t)m * 2 * kGuide;
        const unsigned long long n_ids = TRACE ? (unsigned long long)tp.count
                                               : R.n_run * (unsigned long long)(mp.has_ext + mp.has_point);
        // address of entry c = 0 in the lane's copy of the table; entry c is at tab0 + ES c
        const unsigned tab0 = (unsigned)__cvta_generic_to_shared(s_tab) + 8u * (unsigned)(lane & ((1 << LOGC) - 1)) + ES * (unsigned)ldS;
        const unsigned pa_out = tab0 + ES * (unsigned)(Np + 1);                     // the sentinel beyond the outer surface
        // raw quantum when every package carries the same one
        const unsigned long long q_uni =
            (unsigned long long)__float2ll_rn((mp.has_ext ? mp.qs_ext : mp.qs_point) * R.qscale);

        bool has = false;                            // the lane flies a package (state parked in its slot during events)
        unsigned fslot = 0;                          // the slot of that package
        unsigned long long ch_next = 0, ch_end = 0;  // warp-uniform id chunk
        bool exhausted = false;
        // flight state: a = +-s along-ray coordinate, positive along the direction of the entry ahead; b2s = impact
        // parameter^2 (units of R^2) with the sign bit set when the next event is an absorption; col = remaining column
        // (units of 1/kappa_ref); pa = shared-memory address of the candidate surface passage
        float a = 0.f, b2s = 0.f, col = 0.f;
        unsigned pa = tab0, pa0 = tab0;

        for (;;) {
            // =====================================================================================
            // EVENT phase: typed batches of up to 32 pending events of the whole pool
            // =====================================================================================
            if (has) {
                sts_f4(aA + 16u * fslot, a, b2s, col, __int_as_float((int)(pa - tab0) >> ESH));
                if (TRACE) { pT[2 * P + (int)fslot] += (int)((pa - pa0) >> ESH); pa0 = pa; }
            }
            __syncwarp();
            int nR;
            for (;;) {
                // lengths of the stacks (lanes that found the ready stack empty have driven its length below zero)
                const uint4 c4 = lds_u4(cq);
                nR = max((int)c4.x, 0);
                const int nA = (int)c4.y, nS = (int)c4.z, nL = (int)c4.w;
                int ft, nq;
                if (nA >= 32) { ft = FQ_ABS; nq = nA; }
                else if (nL >= 32) { ft = FQ_SRC; nq = nL; }
                else if (nS >= 32) { ft = FQ_SCA; nq = nS; }
                else {
                    // partial batches only while too few packages are ready to fly
                    if (nA + nS + nL == 0 || nR >= R.min_ready) break;
                    if (nA >= nS && nA >= nL) { ft = FQ_ABS; nq = nA; }
                    else if (nL >= nS) { ft = FQ_SRC; nq = nL; }
                    else { ft = FQ_SCA; nq = nS; }
                }
                // ---- the batch: the last 32 slots of the stack
                const int cnt = min(nq, 32);
                const bool act = lane < cnt;
                const unsigned slot = act ? lds_u8(qb + (unsigned)(ft * P + nq - 1 - lane)) : 0u;
                const bool issrc = ft == FQ_SRC;

                // ---- the package of the slot
                float es = 0.f, eb2 = 0.f, ecol = 0.f;
                int ec = 1;                                      // entry index of the candidate surface passage
                unsigned blk = 0, kf = 0;
                unsigned long long id = 0, q = q_uni;
                int pkg = 0, n_ev = 0;
                unsigned ncross = 0;
                if (act) {
                    const float4 a4 = lds_f4(aA + 16u * slot);
                    const uint4 b4 = lds_u4(aB + 16u * slot);
                    es = a4.x; eb2 = fabsf(a4.y); ecol = a4.z; ec = __float_as_int(a4.w);
                    id = (unsigned long long)b4.x | ((unsigned long long)b4.y << 32); blk = b4.z; kf = b4.w;
                    if (!R.uniform_q) q = lds_u64(aQ + 8u * slot);
                    if (TRACE) { pkg = pT[slot]; n_ev = pT[P + slot]; ncross = (unsigned)pT[2 * P + slot]; }
                }
                int k = (int)(kf & KF_K);
                bool fly = false, ev_absorb = false;

                if (!issrc) {
                    // ================= absorption + re-emission (L87) or scattering (L85) =================
                    const bool isabs = ft == FQ_ABS;
                    // the flight stopped after committing the passage before entry ec with col < 0: the event lies in
                    // the shell traversed on the way to that surface, col / rho^ before it
                    const int ci = ec - 1;
                    int j = ci <= 0 ? -ci : ci - 1;
                    if (TRACE && act) ncross -= 1u;                                  // the passage beyond the event is none
                    const float s_stop = (ci <= 0) ? -es : es;                      // signed coordinate of that surface
                    unsigned long long old = 0;
                    unsigned peers = 0;
                    int leader = 0;
                    const unsigned actm = __ballot_sync(kFull, act);
                    if (isabs) {
                        // (1) add the package's quantum to the shell tally, keep the old value (L87).  The returning
                        //     atomic is issued here and its result is only needed after the Philox block.
                        if (TRACE) {
                            if (act && MODE == 0) old = gA[j * kTallyStride];
                        } else if (MODE == 1) {
                            if (act) smem_add64(&s_A[j], &s_A[ldS + j], q);
                        } else if (R.uniform_q) {
                            peers = __match_any_sync(kFull, act ? j : -1 - lane);
                            leader = __ffs(peers) - 1;
                            if (act && lane == leader) old = atomicAdd(&gA[j * kTallyStride], q * (unsigned long long)__popc(peers));
                        } else if (act) {
                            old = atomicAdd(&gA[j * kTallyStride], q);
                        }
                        wc_abs += (unsigned)cnt;
                    } else {
                        wc_sca += (unsigned)cnt;
                    }
                    if (act) {
                        uint32_t xw[4];
                        unsigned b = blk;
                        philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), b, (uint32_t)m + R.model0, xw);
                        float u0 = uniform24(xw[0]);
                        if (isabs) {
                            int row;
                            if (MODE == 1) {
                                row = s_row[j];
                            } else {
                                const int hint = s_row[j];
                                if (!TRACE && R.uniform_q)
                                    old = __shfl_sync(actm, old, leader) + q * (unsigned long long)__popc(peers & lt_mask);
                                // emitted power per mass before and after this absorption; rows of the table (R4)
                                const double cs = s_cs[j];
                                const float eps_old = (float)((double)old * cs);
                                const float eps_new = (float)((double)(old + q) * cs);
                                row = row_from(s_eps, nT, hint, eps_old);
                                if (row > hint) atomicMax(&s_row[j], row);
                                const bool same = (row == nT - 1) || (eps_new < s_eps[row]);
                                if (eps_new >= s_eps[nT - 1]) atomicAdd(&s_cnt[LC_CLAMP_HI], 1ull);
                                if (!same) {
                                    // the interval spans table rows: block b gives eps*, the event block is b + 1
                                    const float es_ = eps_old + u0 * (eps_new - eps_old);
                                    row = row_from(s_eps, nT, row, es_);
                                    atomicAdd(&s_cnt[LC_EXTRA_BLOCKS], 1ull);
                                    b++;
                                    philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), b, (uint32_t)m + R.model0, xw);
                                    u0 = uniform24(xw[0]);
                                }
                            }
                            // new frequency bin (L87, R4)
                            k = sample_cdf(D.F + (size_t)row * K, D.guideF + (size_t)row * kGuide, u0);
                        }
                        blk = b + 1u;
                        const float u1 = uniform24(xw[1]);
                        const float tauS = neg_log(uniform24(xw[2]));       // Eq. 1
                        const float tauA = neg_log(uniform24(xw[3]));
                        // ---- event site: the step is truncated where the column ran out (L85 / L87)
                        const float se = s_stop + ecol / fabsf(lds_entry(tab0 + ES * (unsigned)ci).y);
                        const float re2 = fmaf(se, se, eb2);
                        const float re = sqrtf(re2);
                        float mu = 2.f * u1 - 1.f;                          // re-emission: isotropic (L87)
                        if (!isabs) {
                            // ---- scattering with the HG phase function (L85, L167)
                            float mu0 = re > 0.f ? se / re : 1.f;
                            mu0 = fminf(1.f, fmaxf(-1.f, mu0));
                            const float sm = sqrtf(fmaxf(1.f - mu0 * mu0, 0.f));
                            const float ct = hg_cos(s_bin[k].z, u0);
                            const float sth = sqrtf(fmaxf(1.f - ct * ct, 0.f));
                            mu = mu0 * ct + sm * sth * cospif(2.f * u1);
                            mu = fminf(1.f, fmaxf(-1.f, mu));
                        }
                        record<TRACE>(tp, pkg, n_ev, isabs ? 2 /*ABSORB*/ : 1 /*SCATTER*/, j - mp.cav, k, ncross);
                        draw_column(s_bin[k], tauS, tauA, ecol, ev_absorb);
                        // ---- next flight: from shell j towards its inner (s < 0) or outer surface; an impact parameter
                        //      beyond the outer surface of the shell (by rounding only) grazes it
                        es = re * mu;
                        eb2 = fminf(re2 * (1.f - mu) * (1.f + mu), lds_entry(tab0 + ES * (unsigned)(j + 1)).x);
                        ec = (es < 0.f) ? -j : j + 1;
                        fly = true;
                    }
                } else {
                    // ================= escape tally (L87 last sentence) + launch of the next package id (L51-65) ==========
                    const bool esc = act && (kf & KF_OCC);
                    const unsigned escmask = __ballot_sync(kFull, esc);
                    if (escmask) {
                        if (esc) {
                            if (!TRACE) smem_add64(&s_esc[k], &s_esc[K + k], q);
                            record<TRACE>(tp, pkg, n_ev, 3 /*ESCAPE*/, D.N - 1, k, ncross);
                            if (TRACE) tp.n_events[pkg] = n_ev;
                        }
                        wc_esc += __popc(escmask);
                    }
                    unsigned long long inj = 0;                  // raw units injected by this lane (per-package quanta)
                    bool need = act;
                    while (__any_sync(kFull, need) && !exhausted) {
                        // free slots take the next package id from the global counter
                        bool launch = false;
                        const unsigned needmask = __ballot_sync(kFull, need);
                        {
                            const unsigned cntn = __popc(needmask);
                            const unsigned rank = __popc(needmask & lt_mask);
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
                                if (need && rank >= avail) {
                                    jdx = base + (rank - avail);
                                    got = jdx < nend;
                                }
                                ch_next = base + (cntn - avail);
                                if (ch_next > nend) ch_next = nend;
                                ch_end = nend;
                            }
                            if (got) {
                                if (TRACE) {
                                    pkg = (int)jdx;
                                    id = tp.first_id + jdx;
                                } else {
                                    // run-local index -> source and global package id (R2)
                                    const bool second = jdx >= R.n_run;
                                    id = (second ? R.n_total + (jdx - R.n_run) : jdx) + R.id_base;
                                }
                                launch = true;
                            }
                            wc_pkg += __popc(__ballot_sync(kFull, launch));
                        }
                        need = false;
                        if (launch) {
                            // ---- launch: one Philox block
                            uint32_t xw[4];
                            const bool point = mp.has_ext ? ((id - R.id_base) >= R.n_total) : true;
                            philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), 0u, (uint32_t)m + R.model0, xw);
                            blk = 1u;
                            const float u0 = uniform24(xw[0]), u1 = uniform24(xw[1]);
                            k = sample_cdf(g_src + (point ? K : 0), g_srcguide + (point ? kGuide : 0), u0);   // L55
                            float re, re2, mu, b2src = 0.f, w = 1.f;
                            int j;
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
                            ncross = 0; n_ev = 0;
                            q = (unsigned long long)__float2ll_rn(w * (point ? mp.qs_point : mp.qs_ext) * R.qscale);
                            inj += q;                                // (FFI splits the quantum below)
                            record<TRACE>(tp, pkg, n_ev, 0 /*LAUNCH*/, j - mp.cav, k, 0);
                            fly = true;
                            if (R.ffi) {
                                // forced first interaction (Eq. 9-12, R11).  The optical depth tau0 of the whole launch chord is
                                // summed here, in the launch batch, with the arithmetic of the crossing step
                                float cdry = mp.colmax;
                                {
                                    const float sw = re * mu;
                                    float b2w = point ? re2 * (1.f - mu) * (1.f + mu) : b2src;
                                    unsigned pw = tab0 + ES * (unsigned)((sw < 0.f) ? -j : j + 1);
                                    float aw = (pw <= tab0) ? -sw : sw;
                                    unsigned nff = 0;
                                    for (;;) {
                                        const float2 T = lds_entry(pw);
                                        const float d = T.x - b2w;
                                        if (d >= 0.f) {
                                            const float t = fmaf(T.y, aw, cdry);
                                            aw = sqrt_ftz(d);
                                            cdry = fmaf(-T.y, aw, t);
                                            pw += ES;
                                            nff++;
                                        } else if (pw <= tab0) {
                                            pw = 2u * tab0 + ES - pw;        // tangent shell: on to the mirrored outward entry
                                            aw = -aw;
                                        } else if (pw != pa_out) {
                                            b2w = T.x;                       // graze
                                        } else {
                                            break;                           // the sentinel: the chord has left the model
                                        }
                                    }
                                    lc_ffi += nff;
                                }
                                const float kext = s_bin[k].w;
                                const float tau0 = kext * (mp.colmax - cdry);          // Eq. 9
                                const float Pint = -expm1f(-tau0);                     // Eq. 12
                                const unsigned long long q_un = min(q, (unsigned long long)__float2ll_rn((float)q * expf(-tau0)));
                                if (!TRACE && q_un) smem_add64(&s_esc[k], &s_esc[K + k], q_un);   // un-interacted share escapes in bin k
                                q -= q_un;
                                if (!(tau0 > 0.f)) {
                                    atomicAdd(&s_cnt[LC_UNINTERACTED], 1ull);
                                    record<TRACE>(tp, pkg, n_ev, 5 /*UNINTERACTED*/, j - mp.cav, k, 0);
                                    if (TRACE) tp.n_events[pkg] = n_ev;
                                    fly = false; need = true;            // the slot takes another package id
                                } else {
                                    const float tauE = -log1pf(-uniform24(xw[2]) * Pint);  // Eq. 10
                                    ev_absorb = !(uniform24(xw[3]) < s_omega[k]);
                                    ecol = tauE / kext;
                                }
                            } else {
                                draw_column(s_bin[k], neg_log(uniform24(xw[2])), neg_log(uniform24(xw[3])), ecol, ev_absorb);
                            }
                            // ---- first flight: from shell j towards its inner (s < 0) or outer surface
                            es = re * mu;
                            eb2 = point ? re2 * (1.f - mu) * (1.f + mu) : b2src;
                            ec = (es < 0.f) ? -j : j + 1;
                        }
                    }
                    if (!R.uniform_q) {
                        const unsigned lm = __ballot_sync(kFull, inj != 0ull);
                        if (lm) {
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) inj += __shfl_xor_sync(kFull, inj, o);
                            if (lane == 0) atomicAdd(&s_cnt[LC_INJECTED_RAW], inj);
                        }
                    }
                }
                // ---- the package goes back into its slot and onto the ready stack; a slot that got no package id
                //      (the ids of the ticket are exhausted) leaves the pool
                const unsigned flym = __ballot_sync(kFull, fly);
                if (fly) {
                    const float b2w = __uint_as_float(__float_as_uint(eb2) | (ev_absorb ? 0x80000000u : 0u));
                    sts_f4(aA + 16u * slot, fabsf(es), b2w, ecol, __int_as_float(ec));
                    sts_u4(aB + 16u * slot, (unsigned)id, (unsigned)(id >> 32), blk, (unsigned)k | KF_OCC);
                    if (!R.uniform_q) sts_u64(aQ + 8u * slot, q);
                    if (TRACE) { pT[slot] = pkg; pT[P + slot] = n_ev; pT[2 * P + slot] = (int)ncross; }
                    sts_u8(qb + (unsigned)(nR + __popc(flym & lt_mask)), slot);
                }
                if (lane == 0) {
                    sts_u32(cq, (unsigned)(nR + __popc(flym)));
                    sts_u32(cq + 4u * (unsigned)ft, (unsigned)(nq - cnt));
                }
                __syncwarp();
            }
            // every slot of the pool has left it: the ticket is drained
            if (nR == 0 && !__any_sync(kFull, has)) break;
            if (lane == 0) sts_u32(cq, (unsigned)nR);                // (a length below zero starts again at zero)
            __syncwarp();

            // =====================================================================================
            // CROSSING phase (Eq. 4): no RNG, no global memory, no branches in the crossing itself.
            // One crossing: d = r_c^2 - b^2 (negative: the surface is not reached, the lane stops with col
            // untouched); along-ray coordinate of the surface sn = +-sqrt(d); col -= rho^ (sn - s) (Eq. 4) is
            // committed together with the passage, and the lane stops if col < 0: the event lies col / rho^
            // before the surface (R7: an event exactly on a surface is a passage).
            // =====================================================================================
            if (has) {
                const float4 a4 = lds_f4(aA + 16u * fslot);
                a = a4.x; b2s = a4.y; col = a4.z; pa = tab0 + ES * (unsigned)__float_as_int(a4.w);
            }
            for (int it = 0; it < R.visit; it++) {
                // ---- a lane without a flight pops the ready stack (a length that has reached zero goes on falling)
                if (!has) {
                    const int idx = (int)atoms_add(cq, 0xffffffffu) - 1;
                    if (idx >= 0) {
                        fslot = lds_u8(qb + (unsigned)idx);
                        const float4 a4 = lds_f4(aA + 16u * fslot);
                        a = a4.x; b2s = a4.y; col = a4.z; pa = tab0 + ES * (unsigned)__float_as_int(a4.w);
                        pa0 = pa;
                        has = true;
                    }
                }
                // ---- kSteps crossings.  The table is walked from pb with constant offsets; the entries are read two
                //      steps ahead of their use and unconditionally (a lane that has stopped reads on harmlessly), so
                //      that no crossing waits for a shared-memory load
                const unsigned pb = pa;
                const float b2 = fabsf(b2s);
                bool alive = has;
                float2 T0 = lds_entry(pb), T1 = lds_entry(pb + ES);
#pragma unroll
                for (int u = 0; u < kSteps; u++) {
                    const float2 T2 = lds_entry(pb + ES * (u + 2));
                    const float d = T0.x - b2;
                    alive = alive && (d >= 0.f);
                    if (alive) {
                        // col -= rho^ (sn - s) as (col + rho^ s) - rho^ sn with s = +-a, sn = +-sqrt(d), T0.y = +-rho^
                        const float t = fmaf(T0.y, a, col);
                        a = sqrt_ftz(d);
                        col = fmaf(-T0.y, a, t);
                        pa += ES;
                    }
                    alive = alive && (col >= 0.f);
                    T0 = T1; T1 = T2;
                }
                lc8 += pa - pb;
                // ---- block end.  A lane that stopped short of an inward surface with column left is in its tangent
                //      shell: it heads for the outer surface instead, entry c -> entry 1 - c (the 1 - 2c entries skipped
                //      are no passages), the coordinate now runs along an outward entry.  Every other stop ends the
                //      flight: the column ran out (scattering or absorption) or the sentinel was reached (escape).
                const bool colpos = col >= 0.f;
                const bool tang = has && !alive && colpos && (pa <= tab0);
                if (tang) {
                    const unsigned np = 2u * tab0 + ES - pa;
                    if (TRACE) pa0 += np - pa;
                    pa = np;
                    a = -a;
                }
                if (has && !alive && !tang) {
                    sts_f4(aA + 16u * fslot, a, b2s, col, __int_as_float((int)(pa - tab0) >> ESH));
                    const unsigned ft = colpos ? (unsigned)FQ_SRC : ((__float_as_int(b2s) < 0) ? (unsigned)FQ_ABS : (unsigned)FQ_SCA);
                    const unsigned pos = atoms_add(cq + 4u * ft, 1u);
                    sts_u8(qb + ft * (unsigned)P + pos, fslot);
                    if (TRACE) pT[2 * P + (int)fslot] += (int)((pa - pa0) >> ESH);
                    has = false;
                }
            }
            __syncwarp();
            // counters: flush before a 32-bit count can wrap
            if (__any_sync(kFull, ((lc8 >> 2) | lc_ffi | wc_pkg | wc_sca | wc_abs | wc_esc) >> 29) != 0u) {
                atomicAdd(&s_cnt[LC_CROSSINGS], (unsigned long long)(lc8 >> ESH));
                if (lc_ffi) atomicAdd(&s_cnt[LC_FFI_CROSSINGS], (unsigned long long)lc_ffi);
                if (lane == 0) {
                    atomicAdd(&s_cnt[LC_PACKAGES], (unsigned long long)wc_pkg);
                    atomicAdd(&s_cnt[LC_SCATTERINGS], (unsigned long long)wc_sca);
                    atomicAdd(&s_cnt[LC_ABSORPTIONS], (unsigned long long)wc_abs);
                    atomicAdd(&s_cnt[LC_ESCAPED], (unsigned long long)wc_esc);
                    // the passage committed beyond an event site is none: one per event that has been handled so far
                    atomicAdd(&s_cnt[LC_CROSSINGS], 0ull - (unsigned long long)(wc_sca + wc_abs));
                    if (R.uniform_q) atomicAdd(&s_cnt[LC_INJECTED_RAW], q_uni * (unsigned long long)wc_pkg);
                }
                lc8 = lc_ffi = wc_pkg = wc_sca = wc_abs = wc_esc = 0u;
            }
        }
        // ---------------- per-ticket flush of the warp's counts (identical quanta: injected raw units = launches x quantum)
        {
            unsigned long long c = lc8 >> ESH, f = lc_ffi;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { c += __shfl_xor_sync(kFull, c, o); f += __shfl_xor_sync(kFull, f, o); }
            if (lane == 0) {
                atomicAdd(&s_cnt[LC_CROSSINGS], c - (unsigned long long)(wc_sca + wc_abs));
                if (f) atomicAdd(&s_cnt[LC_FFI_CROSSINGS], f);
                atomicAdd(&s_cnt[LC_PACKAGES], (unsigned long long)wc_pkg);
                atomicAdd(&s_cnt[LC_SCATTERINGS], (unsigned long long)wc_sca);
                atomicAdd(&s_cnt[LC_ABSORPTIONS], (unsigned long long)wc_abs);
                atomicAdd(&s_cnt[LC_ESCAPED], (unsigned long long)wc_esc);
                if (R.uniform_q) atomicAdd(&s_cnt[LC_INJECTED_RAW], q_uni * (unsigned long long)wc_pkg);
            }
            lc8 = lc_ffi = wc_pkg = wc_sca = wc_abs = wc_esc = 0u;
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
                if (v) atomicAdd(&gA[x * kTallyStride], v);
            }
    }

    if (TRACE) return;
    // ---------------- counters: one atomic per block and counter
    __syncthreads();
    if (tid < LC_N && s_cnt[tid]) atomicAdd(&D.counters[tid], s_cnt[tid]);
}

}  // namespace dies
