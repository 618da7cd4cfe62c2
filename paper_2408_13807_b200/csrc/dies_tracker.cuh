// dies_tracker.cuh -- the persistent-thread IRE package tracker for sm_100a (hot path of include/dies.h).
//
// Every warp owns a POOL of P photon packages whose state lives in shared memory (40 bytes per package) and four
// small queues of pool slots: packages ready to fly, and packages waiting for an absorption, a scattering, or a
// source event (escape tally + launch of the next package id).  The warp alternates
// between
//   (1) a CROSSING phase: 32 flying packages in registers run the shell-crossing loop (Eq. 4) with
//       no random numbers, no global memory and no branches (every crossing is predicated on the lane still flying).
//       When fewer than thr_hi lanes still fly, the stopped lanes write their package back, queue it by event type
//       and take the next ready package from the pool, so the loop keeps (nearly) all lanes busy until the ready
//       queue is empty;
//   (2) an EVENT phase: batches of 32 queued events, of ONE type whenever a queue holds 32 (mixed only when the
//       crossing phase would starve), run one shared instruction stream: escapes are tallied, new package ids taken
//       from the model's global counter, absorptions update the 64-bit fixed-point shell tallies (one returning
//       atomic per distinct shell in the warp, issued before and consumed after the Philox block), then a
//       Philox4x32-10 block, two new free paths (Eq. 1), the table search for the new frequency, the new
//       direction and the set-up of the next flight.
// Differences from the paper's OpenCL design are listed in DESIGN.md ("What differs from the paper").
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dies {

constexpr int kBlock = 256;          // threads per block
constexpr int kWarps = kBlock / 32;
constexpr int kMinBlocks = 4;        // resident blocks per SM asked from the compiler (64 registers)
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kChunk = 128;     // package ids a warp takes from the global counter at a time (large runs)
constexpr int kUnroll = 12;           // crossings per vote in the crossing loop
constexpr int kMaxPool = 248;        // pool slots per warp (queue entries are bytes)
constexpr int kGuide = 1024;         // cut-points per CDF row of the guide tables
constexpr int kTallyStride = 32;     // 64-bit words between the absorbed-energy tallies of two shells: one tally per
                                     // 256 bytes, because the L2 atomic unit serialises updates of the same line

// event counters (same order as DIES_C_* in include/dies.h), accumulated per block in shared memory
enum { LC_PACKAGES = 0, LC_CROSSINGS, LC_FFI_CROSSINGS, LC_SCATTERINGS, LC_ABSORPTIONS, LC_ESCAPED, LC_UNINTERACTED,
       LC_TERMINATED, LC_EXTRA_BLOCKS, LC_CLAMP_HI, LC_INJECTED_RAW, LC_TERMINATED_RAW, LC_REWEIGHT_RAW, LC_N };

// per-slot flag word: frequency bin | type of the pending event | slot holds a package
constexpr unsigned KF_K = 0xffffu, KF_EVABS = 1u << 16, KF_OCC = 1u << 18;
// the queues of a warp
enum { QT_ABS = 0, QT_SCA, QT_SRC, QT_READY, QT_N };

struct ModelParams {
    int Np;            // internal shells = n_shells + cav
    int cav;           // 1 if r_bounds[0] > 0: internal shell 0 is the empty cavity (R10)
    int has_ext, has_point;
    float r0hat;       // r_bounds[0] / R
    float qs_ext, qs_point;   // e_src / e_ref (<= 1): raw units per unit-weight package / 2^S
    float colmax;      // a column (units of 1/kappa_ref) larger than that of any chord: start value of the FFI chord sum
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
    const unsigned short* guideF;    // nT x kGuide: smallest k with F[t][k] > c / kGuide
    const unsigned short* guideS;    // n_models x 2 x kGuide: the same for the source CDFs
    const float2* stab;              // n_models x ldT unfolded shell table
    const float4* stabW;             // the same for a run with free-path weighting: {r^2, +-rho^, k_A rho^, k_A}
    const double* cscale;            // n_models x ldS: eps^ per raw tally unit
    const float* srccdf;             // n_models x 2 x K: external, point
    const ModelParams* mp;           // n_models
    const int* fixed_row;            // n_models x ldS
    unsigned long long* A;           // n_models x ldS x kTallyStride: absorbed-energy tallies (raw fixed point), strided
    unsigned long long* esc;         // n_models x K     escape tallies (raw fixed point)
    unsigned long long* next_id;     // n_models         run-local package counter
    unsigned long long* counters;    // DIES_N_COUNTERS
    unsigned int* ticket;            // 1
};

// shared-memory plan of a block (byte offsets), used by the kernel and by the host to size the launch
struct SmemPlan { unsigned bin, cs, tab, eps, omega, row, esc, A, poolA, poolB, poolQ, poolW, queues, trace, total; };
__host__ __device__ inline SmemPlan plan_smem(int K, int nT, int ldS, int ldT, int P, bool trace, bool with_q,
                                              bool wt = false)
{
    SmemPlan p;
    unsigned o = 0;
    p.bin = o;   o += 16u * K;                       // float4 K
    p.cs = o;    o += 8u * ldS;                      // double ldS
    p.cs = (p.cs + 15u) & ~15u; o = p.cs + 8u * ldS; o = (o + 15u) & ~15u;
    p.tab = o;   o += (wt ? 16u : 8u) * ldT;         // float2 (float4 with free-path weighting) ldT
    p.eps = o;   o += 4u * nT;
    p.omega = o; o += 4u * K;
    p.row = o;   o += 4u * ldS;
    p.esc = o;   o += 8u * K;                        // low words, high words
    p.A = o;     o += 8u * ldS;                      // low words, high words (fixed-T mode)
    o = (o + 15u) & ~15u;
    p.poolA = o; o += 16u * kWarps * P;              // float4 {s, b2, col, pa}
    p.poolB = o; o += 16u * kWarps * P;              // uint4  {id lo, id hi, blk, flags}
    p.poolQ = o; if (with_q) o += 8u * kWarps * P;   // raw quantum of the package (not stored when all are equal)
    o = (o + 15u) & ~15u;
    p.poolW = o; if (wt) o += 16u * kWarps * P;      // float4 {colS, colA at the draw, colS at the draw, launch quantum}
    p.queues = o; o += (unsigned)(QT_N * kWarps * P);
    o = (o + 15u) & ~15u;
    p.trace = o; if (trace) o += 12u * kWarps * P;   // pkg, n_ev, crossings so far
    p.total = o;
    return p;
}

struct RunParams {
    unsigned long long n_run;        // packages per source in this call
    unsigned long long id_base;      // packages per source done by earlier calls (accumulate)
    unsigned long long n_total;      // packages per source over the whole run
    uint32_t key0, key1;
    uint32_t model0;                 // index of the handle's first model in the Philox counter (a shard of a batch)
    uint32_t rk[20];                 // Philox round keys: rk[2r] = key0 + r 0x9E3779B9, rk[2r+1] = key1 + r 0xBB67AE85
    float k_bg;
    int ffi;
    int uniform_q;                   // all packages carry the same raw quantum (no k_bg, no FFI, one source)
    int weighted;                    // free-path weighting (Eq. 8, R17): two clocks, package weights change in flight
    float k_S;                       // scattering clock factor
    double k_A, k_A_dilute;          // absorption clock factor(s) (host side: they go into stabW)
    float g_E, g_S;                  // directional weighting of re-emission (Eq. 6) and scattering (Eq. 7); R19
    int use_gS;                      // Eq. 7 active (g_S = 0 is a weighting too)
    int reemit_cell;                 // L253 (R20): re-emit from a random position of the cell volume
    float qscale;                    // 2^S
    int n_tickets, parts;            // tickets = n_models * parts
    unsigned chunk;                  // package ids a warp takes at a time: kChunk, fewer (>= 32) when a run is small
    int pool;                        // P: pool slots per warp (multiple of 8, 32 <= P <= kMaxPool)
    int thr_hi;                      // crossing phase: swap stopped lanes for ready packages when fewer fly
    int thr_lo;                      // crossing phase: with no ready package left, leave when fewer fly
    int min_ready;                   // event phase: mixed batches only while fewer packages are ready
    int slots;                       // dies_fly: pool slots per lane (1 <= slots <= kMaxSlots)
    int visit;                       // dies_fly: crossing blocks between two event phases
};

struct TraceParams {
    int model;
    unsigned long long first_id;     // global package id of the first traced package
    int count;
    int32_t* events;                 // count x max_events x 4
    int max_events;
    int32_t* n_events;               // count
    unsigned long long* counter;     // zeroed: next traced package
};

// ------------------------------------------------------------------ RNG contract (include/dies.h)
__device__ __forceinline__ void philox4x32_10_rk(const uint32_t (&rk)[20], uint32_t c0, uint32_t c1, uint32_t c2,
                                                 uint32_t c3, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
        const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r];
        c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
        c3 = (uint32_t)p0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;   // one IMAD.WIDE gives both halves
        const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c3 = (uint32_t)p0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u = ((x >> 9) + 0.5) 2^-23 (R1) without an integer-to-float conversion: 1.m - (1 - 2^-24) is exact
__device__ __forceinline__ float uniform24(uint32_t x)
{
    return __uint_as_float(0x3f800000u | (x >> 9)) - 0.99999994039535522461f;
}

// -ln u for u in (0,1) through the hardware log2 (absolute error of lg2.approx <= 2^-22 on [0.5, 2), 2 ulp elsewhere:
// <= 1.7e-7 in optical depth, the size of the fp32 rounding of the path itself; R14)
__device__ __forceinline__ float neg_log(float u)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(u));
    return y * -0.69314718055994530942f;
}

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

// one 16-byte entry of the unfolded shell table of a run with free-path weighting
__device__ __forceinline__ float4 lds_entry4(unsigned a)
{
    float4 v;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}

// the pool and the queues of a warp are addressed in the shared window directly (32-bit addresses, no generic pointers)
__device__ __forceinline__ unsigned lds_u8(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u8(unsigned a, unsigned v) { asm volatile("st.shared.u8 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ unsigned lds_u32(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(unsigned a, unsigned v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ float4 lds_f4(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_f4(unsigned a, float x, float y, float z, float w)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" :: "r"(a), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
__device__ __forceinline__ uint4 lds_u4(unsigned a)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u4(unsigned a, unsigned x, unsigned y, unsigned z, unsigned w)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" :: "r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ unsigned long long lds_u64(unsigned a)
{
    unsigned long long v;
    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u64(unsigned a, unsigned long long v) { asm volatile("st.shared.u64 [%0], %1;" :: "r"(a), "l"(v) : "memory"); }

// smallest k with cdf[k] > u for a non-decreasing cdf whose last entry exceeds every u (inverse-CDF sampling, R3),
// by the cut-point method: guide[c] is the answer for u = c / kGuide, so the answer for u in [c, c+1) / kGuide is
// found by walking up from it -- one or two table reads instead of a bisection over the whole row
__device__ __forceinline__ int sample_cdf(const float* __restrict__ cdf, const unsigned short* __restrict__ guide, float u)
{
    int k = __ldg(guide + (int)(u * (float)kGuide));
    while (__ldg(cdf + k) <= u) k++;
    return k;
}

// t(eps) = #{j : grid[j] <= eps} clamped to n-1, from a hint t0 near t(eps): the table row of a cell emitting eps
// (R4).  Rows only move up during a run, so the scan from the block's last known row is short.  The hint is shared by
// the warps of a block: a warp whose atomic returned an older (smaller) tally than the one the hint was raised for
// first steps down to its own row.
__device__ __forceinline__ int row_from(const float* grid, int n, int t0, float eps)
{
    int t = t0;
    while (t > 0 && grid[t - 1] > eps) t--;
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

// per-slot trace state (TRACE kernels only): pkg, number of events so far, crossings so far
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
// TRACE : replay tp.count packages of one model, tallies read-only, events recorded
// WT    : free-path weighting (Eq. 8; R17): absorption and scattering clocks are kept
//         apart (they run k_A,i and k_S times faster than the true optical depths), the package quantum follows Eq. 8
template <int MODE, bool TRACE, bool WT>
__global__ void __launch_bounds__(kBlock, kMinBlocks) dies_track(DeviceModel D, RunParams R, TraceParams tp)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = D.K, nT = D.nT, ldS = D.ldS, ldT = D.ldT, P = R.pool;
    const SmemPlan sp = plan_smem(K, nT, ldS, ldT, P, TRACE, !R.uniform_q, WT);
    constexpr unsigned ES = WT ? 16u : 8u;           // bytes per entry of the unfolded shell table
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
    // the pool and the queues of this warp
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem_raw);
    const unsigned aA = sbase + sp.poolA + 16u * (unsigned)(wid * P);          // float4 {s, b2, col, pa} per slot
    const unsigned aB = sbase + sp.poolB + 16u * (unsigned)(wid * P);          // uint4 {id lo, id hi, blk, flags}
    const unsigned aQ = sbase + sp.poolQ + 8u * (unsigned)(wid * P);           // raw quantum
    const unsigned aW = sbase + sp.poolW + 16u * (unsigned)(wid * P);          // WT: second clock and the draw
    const unsigned qA = sbase + sp.queues + (unsigned)(wid * QT_N * P);        // byte queues of pool slots
    const unsigned qS = qA + (unsigned)P, qL = qS + (unsigned)P, qR = qL + (unsigned)P;
    int* const pT = reinterpret_cast<int*>(smem_raw + sp.trace) + wid * 3 * P;      // TRACE only

    for (int x = tid; x < K; x += kBlock) { s_bin[x] = D.bintab[x]; s_omega[x] = D.omega[x]; }
    for (int x = tid; x < nT; x += kBlock) s_eps[x] = D.epsgrid[x];
    if (tid < LC_N) s_cnt[tid] = 0ull;

    const int thr_hi = R.thr_hi, thr_lo = R.thr_lo, min_ready = R.min_ready;
    // warp-uniform event counts and per-lane crossing counts since the last flush into s_cnt
    unsigned wc_pkg = 0, wc_sca = 0, wc_abs = 0, wc_esc = 0, lc_cross = 0, lc_ffi = 0;

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
        if (WT) { for (int x = tid; x < ldT; x += kBlock) reinterpret_cast<float4*>(s_tab)[x] = D.stabW[(size_t)m * ldT + x]; }
        else { for (int x = tid; x < ldT; x += kBlock) s_tab[x] = D.stab[(size_t)m * ldT + x]; }
        for (int x = tid; x < ldS; x += kBlock) {
            s_cs[x] = D.cscale[(size_t)m * ldS + x];
            s_row[x] = (MODE == 1) ? D.fixed_row[(size_t)m * ldS + x] : 0;
            s_A[x] = 0u; s_A[ldS + x] = 0u;
        }
        for (int x = tid; x < 2 * K; x += kBlock) s_esc[x] = 0u;
        // every slot of the pool is free and waits for a package id
        for (int x = lane; x < P; x += 32) { sts_u8(qL + x, (unsigned)x); sts_u4(aB + 16u * x, 0u, 0u, 0u, 0u); }
        __syncthreads();

        unsigned long long* const gA = D.A + (size_t)m * ldS * kTallyStride;
        unsigned long long* const g_next = TRACE ? tp.counter : D.next_id + m;
        const float* const g_src = D.srccdf + (size_t)m * 2 * K;
        const unsigned short* const g_srcguide = D.guideS + (size_t)m * 2 * kGuide;
        const unsigned long long n_ids = TRACE ? (unsigned long long)tp.count
                                               : R.n_run * (unsigned long long)(mp.has_ext + mp.has_point);
        const unsigned tab0 = (unsigned)__cvta_generic_to_shared(s_tab) + ES * (unsigned)ldS;   // address of entry c = 0
        const unsigned pa_out = tab0 + ES * (unsigned)(Np + 1);                     // the sentinel beyond the outer surface
        // raw quantum when every package carries the same one
        const unsigned long long q_uni =
            (unsigned long long)__float2ll_rn((mp.has_ext ? mp.qs_ext : mp.qs_point) * R.qscale);

        int nA = 0, nS = 0, nL = P, nR = 0;          // queue lengths (warp-uniform)
        unsigned long long ch_next = 0, ch_end = 0;  // warp-uniform id chunk
        bool exhausted = false;

        for (;;) {
            // =====================================================================================
            // EVENT phase: batches of up to 32 queued events
            // =====================================================================================
            for (;;) {
                if (nA + nS + nL == 0) break;
                int cA = 0, cS = 0, cL = 0;
                if (nA >= 32) cA = 32;
                else if (nL >= 32) cL = 32;
                else if (nS >= 32) cS = 32;
                else {
                    if (nR >= min_ready) break;                  // enough to fly: let the partial batches grow
                    cA = nA; cS = min(nS, 32 - cA); cL = min(nL, 32 - cA - cS);
                }
                int type = -1;
                unsigned slot = 0;
                {
                    int l = lane;
                    if (l < cA) { type = QT_ABS; slot = lds_u8(qA + (nA - 1 - l)); }
                    else if ((l -= cA) < cS) { type = QT_SCA; slot = lds_u8(qS + (nS - 1 - l)); }
                    else if ((l -= cS) < cL) { type = QT_SRC; slot = lds_u8(qL + (nL - 1 - l)); }
                }
                nA -= cA; nS -= cS; nL -= cL;
                const bool isabs = type == QT_ABS, issca = type == QT_SCA, issrc = type == QT_SRC;
                const bool isev = isabs || issca;

                // ---- the package of the slot
                float s = 0.f, b2 = 0.f, col = 0.f;
                unsigned pa = tab0, blk = 0, kf = 0;
                unsigned long long id = 0, q = q_uni;
                int pkg = 0, n_ev = 0;
                unsigned ncross = 0;
                if (type >= 0) {
                    const float4 a = lds_f4(aA + 16u * slot);
                    const uint4 b = lds_u4(aB + 16u * slot);
                    s = a.x; b2 = a.y; col = a.z; pa = __float_as_uint(a.w);
                    id = (unsigned long long)b.x | ((unsigned long long)b.y << 32); blk = b.z; kf = b.w;
                    if (!R.uniform_q) q = lds_u64(aQ + 8u * slot);
                    if (TRACE) { pkg = pT[slot]; n_ev = pT[P + slot]; ncross = (unsigned)pT[2 * P + slot]; }
                }
                int k = (int)(kf & KF_K);
                const bool esc = issrc && (kf & KF_OCC);

                // (0) free-path weighting (Eq. 8, R17): the quantum the package carries at this event.  Along the
                //     flight the true survival probability over the biased one is e^{kappa_A (CA - C)} for the
                //     absorption clock and e^{kappa_S (k_S - 1) C} for the scattering clock (C: column traversed,
                //     CA: the same weighted with k_A of every shell); the event that ended the flight adds 1/k.
                // The package carries its launch quantum q0 and its weight relative to the launch weight, wrel (fp32);
                // the quantum it adds to a tally is q = round(q0 wrel) (R18).  A quantum that has rounded to nothing
                // does not end the package: it flies on, adding nothing, until the rule of L119 ends it.
                float colS = 0.f, cA0 = 0.f, cS0 = 0.f, wrel = 1.f, off = 0.f;
                unsigned long long q0 = q;
                if (WT) {
                    if (type >= 0) { const float4 w4 = lds_f4(aW + 16u * slot); colS = w4.x; cA0 = w4.y; cS0 = w4.z; wrel = w4.w; }
                    q = (unsigned long long)__double2ll_rn((double)q0 * (double)wrel);
                    long long dq = 0;
                    if (isev || esc) {
                        const float4 bt = s_bin[k];
                        // col, colS: the columns CA, C consumed up to the committed surface; cA0, cS0: where the clocks end
                        float CA = col, C = colS, kdiv = 1.f;
                        if (isev) {
                            const float4 Ep = lds_entry4(pa - 16u);           // the passage that was committed last
                            const float rho = fabsf(Ep.y), rhoA = Ep.z;
                            off = isabs ? (cA0 - col) / rhoA : (cS0 - colS) / rho;   // <= 0: the site lies this far before it
                            CA = fmaf(rhoA, off, col);
                            C = fmaf(rho, off, colS);
                            kdiv = isabs ? Ep.w : R.k_S;
                        }
                        const float kapA = bt.x < 3.0e38f ? 1.f / bt.x : 0.f, kapS = bt.y < 3.0e38f ? 1.f / bt.y : 0.f;
                        const float lnW = fmaf(kapA, CA - C, kapS * (R.k_S - 1.f) * C);
                        wrel *= expf(lnW) / kdiv;
                        const unsigned long long qn = (unsigned long long)__double2ll_rn((double)q0 * (double)wrel);
                        dq = (long long)qn - (long long)q;
                        q = qn;
                    }
                    if (__ballot_sync(kFull, dq != 0)) {
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) dq += __shfl_xor_sync(kFull, dq, o);
                        if (lane == 0) atomicAdd(&s_cnt[LC_REWEIGHT_RAW], (unsigned long long)dq);
                    }
                }

                // (1) absorptions first: add the package's quantum to the shell tally, keep the old value (L87).
                //     The returning atomic is issued here and its result is only needed after the Philox block.
                // shell of the event: the one traversed on the way to the surface entry before pa, which was not reached
                const int ci = (int)(pa - tab0) / (int)ES - 1;
                int j = ci <= 0 ? -ci : ci - 1;
                const unsigned absmask = __ballot_sync(kFull, isabs);
                unsigned long long old = 0;
                unsigned peers = 0;
                int leader = 0;
                if (absmask) {
                    if (TRACE) {
                        if (isabs && MODE == 0) old = gA[j * kTallyStride];
                    } else if (MODE == 1) {
                        if (isabs) smem_add64(&s_A[j], &s_A[ldS + j], q);
                    } else if (R.uniform_q) {
                        // the leader's atomic is issued now; its value is broadcast only where the rows are needed, after
                        // the Philox block, so that nothing waits for L2 here
                        peers = __match_any_sync(kFull, isabs ? j : -1 - lane);
                        leader = __ffs(peers) - 1;
                        if (isabs && lane == leader) old = atomicAdd(&gA[j * kTallyStride], q * (unsigned long long)__popc(peers));
                    } else if (isabs) {
                        old = atomicAdd(&gA[j * kTallyStride], q);
                    }
                    wc_abs += (unsigned)cA;
                }
                wc_sca += (unsigned)cS;

                // (2) escapes (PAPER.md L87 last sentence)
                const unsigned escmask = __ballot_sync(kFull, esc);
                if (escmask) {
                    if (esc) {
                        if (!TRACE) smem_add64(&s_esc[k], &s_esc[K + k], q);
                        record<TRACE>(tp, pkg, n_ev, 3 /*ESCAPE*/, D.N - 1, k, ncross);
                        if (TRACE) tp.n_events[pkg] = n_ev;
                    }
                    wc_esc += __popc(escmask);
                }
                // (3) free slots take the next package id from the global counter
                bool launch = false;
                const bool need = issrc;
                const unsigned needmask = __ballot_sync(kFull, need);
                if (needmask && !exhausted) {
                    const unsigned cnt = __popc(needmask);
                    const unsigned rank = __popc(needmask & lt_mask);
                    const unsigned long long avail = ch_end - ch_next;
                    unsigned long long jdx = ch_next + rank;
                    bool got = need && (rank < avail);
                    if (avail >= cnt) {
                        ch_next += cnt;
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
                        ch_next = base + (cnt - avail);
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
                        blk = 0;
                    }
                    wc_pkg += __popc(__ballot_sync(kFull, launch));
                }

                // (4) events: launch / scatter / absorb + re-emit; one Philox block each
                //     (DESIGN.md RNG contract), one instruction stream for all of them
                bool fly = false, ev_absorb = false, uninter = false;
                unsigned long long q_inj = 0;
                if (launch || isev) {
                    uint32_t xw[4];
                    const bool atsrc = launch;                                      // the event site is the source
                    const bool point = atsrc && (mp.has_ext ? ((id - R.id_base) >= R.n_total) : true);
                    unsigned b = blk;
                    philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), b, (uint32_t)m + R.model0, xw);
                    const float* cdf = nullptr;      // table the new frequency bin is drawn from (launch, re-emission)
                    const unsigned short* guide = nullptr;
                    if (isabs) {
                        int row;
                        if (MODE == 1) {
                            row = s_row[j];
                        } else {
                            const int hint = s_row[j];
                            if (!TRACE && R.uniform_q)
                                old = __shfl_sync(absmask, old, leader) + q * (unsigned long long)__popc(peers & lt_mask);
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
                                const float es = eps_old + uniform24(xw[0]) * (eps_new - eps_old);
                                row = row_from(s_eps, nT, row, es);
                                atomicAdd(&s_cnt[LC_EXTRA_BLOCKS], 1ull);
                                b++;
                                philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), b, (uint32_t)m + R.model0, xw);
                            }
                        }
                        cdf = D.F + (size_t)row * K;
                        guide = D.guideF + (size_t)row * kGuide;
                    } else if (launch) {
                        cdf = g_src + (point ? K : 0);                              // L55 source spectrum table
                        guide = g_srcguide + (point ? kGuide : 0);
                    }
                    blk = b + 1u;
                    const float u0 = uniform24(xw[0]), u1 = uniform24(xw[1]);
                    const float tauS = neg_log(uniform24(xw[2]));       // Eq. 1
                    const float tauA = neg_log(uniform24(xw[3]));
                    // new frequency bin (launch: L55; re-emission: L87, R4)
                    if (cdf) k = sample_cdf(cdf, guide, u0);

                    // ---- event site (radius re, re2 = re^2, shell j) and new direction cosine mu w.r.t. the radius
                    float re, re2, mu, b2src = 0.f, wdir = 1.f;
                    fly = true;
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
                            ncross = 0; n_ev = 0;
                            q = (unsigned long long)__float2ll_rn(w * (point ? mp.qs_point : mp.qs_ext) * R.qscale);
                            q0 = q; wrel = 1.f;
                            q_inj = q;                           // (FFI splits the quantum below)
                            record<TRACE>(tp, pkg, n_ev, 0 /*LAUNCH*/, j - mp.cav, k, 0);
                        }
                    } else {
                        // ---- the step is truncated where the column ran out (L85 / L87): the surface passage
                        //      before pa was committed with col < 0, so the site lies col / rho^ before it
                        const float se = WT ? s + off : s + col / fabsf(lds_entry(pa - 8u).y);
                        re2 = fmaf(se, se, b2);
                        re = sqrtf(re2);
                        if (WT && isabs && R.reemit_cell) {
                            // L253 (R20): the package is re-emitted from a radius uniform in the volume of shell j;
                            // one more Philox block gives the uniform
                            uint32_t xr[4];
                            philox4x32_10_rk(R.rk, (uint32_t)id, (uint32_t)(id >> 32), blk++, (uint32_t)m + R.model0, xr);
                            const float ri2 = lds_entry4(tab0 + 16u * (unsigned)j).x, ro2 = lds_entry4(tab0 + 16u * (unsigned)(j + 1)).x;
                            const float ri = sqrtf(ri2), ro = sqrtf(ro2);
                            const float ri3 = ri * ri2, ro3 = ro * ro2;
                            re = cbrtf(fmaf(uniform24(xr[0]), ro3 - ri3, ri3));
                            re = fminf(ro, fmaxf(ri, re));
                            re2 = re * re;
                        }
                        mu = 2.f * u1 - 1.f;             // re-emission: isotropic (L87)
                        // directional weighting (Eq. 6-7, R19) measures angles from the direction towards the centre
                        // for packages of the external field and away from it for those of the central source (L109)
                        const bool ptpkg = mp.has_ext ? ((id - R.id_base) >= R.n_total) : true;
                        if (WT && isabs && R.g_E != 0.f) {
                            // Eq. 6: HG(g_E) instead of isotropic; weight = (1/2) / p_HG(mu')
                            const float mup = hg_cos(R.g_E, u1);
                            const float x = fmaf(-2.f * R.g_E, mup, 1.f + R.g_E * R.g_E);
                            wdir = x * sqrtf(x) / (1.f - R.g_E * R.g_E);
                            mu = ptpkg ? mup : -mup;
                        }
                        if (issca) {
                            // ---- scattering with the HG phase function (L85, L167)
                            float mu0 = re > 0.f ? se / re : 1.f;
                            mu0 = fminf(1.f, fmaxf(-1.f, mu0));
                            const float sm = sqrtf(fmaxf(1.f - mu0 * mu0, 0.f));
                            if (WT && R.use_gS) {
                                // Eq. 7: direction from HG(g_S) about the radial reference direction, azimuth uniform;
                                // weight = dust HG density at the true scattering angle / sampling density
                                const float mup = hg_cos(R.g_S, u0);
                                const float mu1 = ptpkg ? mup : -mup;
                                float ct = mu0 * mu1 + sm * sqrtf(fmaxf(1.f - mu1 * mu1, 0.f)) * cospif(2.f * u1);
                                ct = fminf(1.f, fmaxf(-1.f, ct));
                                const float g = s_bin[k].z;
                                const float xa = fmaf(-2.f * g, ct, 1.f + g * g);
                                const float xb = fmaf(-2.f * R.g_S, mup, 1.f + R.g_S * R.g_S);
                                wdir = ((1.f - g * g) * xb * sqrtf(xb)) / ((1.f - R.g_S * R.g_S) * xa * sqrtf(xa));
                                mu = mu1;
                            } else {
                                const float ct = hg_cos(s_bin[k].z, u0);
                                const float sth = sqrtf(fmaxf(1.f - ct * ct, 0.f));
                                mu = mu0 * ct + sm * sth * cospif(2.f * u1);
                                mu = fminf(1.f, fmaxf(-1.f, mu));
                            }
                        }
                        record<TRACE>(tp, pkg, n_ev, issca ? 1 /*SCATTER*/ : 2 /*ABSORB*/, j - mp.cav, k, ncross);
                    }
                    // ---- column (in units of 1/kappa_ref) to the next event and its type
                    if (R.ffi && atsrc) {
                        // forced first interaction (Eq. 9-12, R11).  The optical depth tau0 of the whole launch chord is
                        // summed here, in the launch batch (all lanes walk their chords together: no exchange, no vote,
                        // no second event for the package), with the arithmetic of the crossing step
                        float cdry = mp.colmax;
                        if (!WT) {
                            const float sw = re * mu;
                            float b2w = point ? re2 * (1.f - mu) * (1.f + mu) : b2src;
                            unsigned pw = tab0 + 8u * (unsigned)((sw < 0.f) ? -j : j + 1);
                            float aw = (pw <= tab0) ? -sw : sw;
                            unsigned nff = 0;
                            for (;;) {
                                const float2 T = lds_entry(pw);
                                const float d = T.x - b2w;
                                if (d >= 0.f) {
                                    const float t = fmaf(T.y, aw, cdry);
                                    aw = sqrt_ftz(d);
                                    cdry = fmaf(-T.y, aw, t);
                                    pw += 8u;
                                    nff++;
                                } else if (pw <= tab0) {
                                    pw = 2u * tab0 + 8u - pw;        // tangent shell: on to the mirrored outward entry
                                    aw = -aw;
                                } else if (pw != pa_out) {
                                    b2w = T.x;                       // graze
                                } else {
                                    break;                           // the sentinel: the chord has left the model
                                }
                            }
                            lc_ffi += nff;
                        }
                        {
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
                                fly = false; uninter = true;
                            } else {
                                const float tauE = -log1pf(-uniform24(xw[2]) * Pint);  // Eq. 10
                                ev_absorb = !(uniform24(xw[3]) < s_omega[k]);
                                col = tauE / kext;
                            }
                        }
                    } else {
                        // L85/L87; R7 tie -> absorption; R15 one column instead of two clocks
                        const float4 bt = s_bin[k];
                        const float cA_ = tauA * bt.x, cS_ = tauS * bt.y;
                        if (WT) {
                            // two clocks counting up from zero: absorption ends at cA0 of k_A-weighted column,
                            // scattering at cS0 of plain column (its factor k_S sits in cS0)
                            cA0 = cA_; cS0 = cS_ / R.k_S;
                            col = 0.f; colS = 0.f;
                        } else {
                            ev_absorb = (cA_ <= cS_);
                            col = fminf(cA_, cS_);
                        }
                    }
                    if (WT && (R.g_E != 0.f || R.use_gS)) {
                        // the quantum the package carries away from a reweighted direction
                        long long dq = 0;
                        if (wdir != 1.f) {
                            wrel *= wdir;
                            const unsigned long long qn = (unsigned long long)__double2ll_rn((double)q0 * (double)wrel);
                            dq = (long long)qn - (long long)q;
                            q = qn;
                        }
                        if (dq != 0) atomicAdd(&s_cnt[LC_REWEIGHT_RAW], (unsigned long long)dq);
                    }
                    // L119: a package whose weight fell by ten orders of magnitude is terminated
                    if (WT && isev && wrel < 1e-10f) {
                        record<TRACE>(tp, pkg, n_ev, 4 /*TERMINATE*/, j - mp.cav, k, ncross);
                        if (TRACE) tp.n_events[pkg] = n_ev;
                        atomicAdd(&s_cnt[LC_TERMINATED], 1ull);
                        if (q) atomicAdd(&s_cnt[LC_TERMINATED_RAW], q);
                        fly = false; uninter = true;
                    }
                    // ---- next flight: from shell j towards its inner (s < 0) or outer surface
                    s = re * mu;
                    b2 = (atsrc && !point) ? b2src : re2 * (1.f - mu) * (1.f + mu);
                    pa = tab0 + ES * (unsigned)((s < 0.f) ? -j : j + 1);
                }
                // ---- write the package back; flying packages join the ready queue, a slot whose package ended
                //      without escaping through the sentinel (FFI, tau0 = 0) is free again; a slot that got no id dies
                if (fly || uninter) {
                    const unsigned nkf = uninter ? 0u
                        : ((unsigned)k | (ev_absorb ? KF_EVABS : 0u) | KF_OCC);
                    sts_f4(aA + 16u * slot, s, b2, col, __uint_as_float(pa));
                    sts_u4(aB + 16u * slot, (unsigned)id, (unsigned)(id >> 32), blk, nkf);
                    if (!R.uniform_q) sts_u64(aQ + 8u * slot, WT ? q0 : q);
                    if (WT) sts_f4(aW + 16u * slot, colS, cA0, cS0, wrel);
                    if (TRACE) { pT[slot] = pkg; pT[P + slot] = n_ev; pT[2 * P + slot] = (int)ncross; }
                }
                if (!R.uniform_q) {
                    // raw units injected by the launches of this batch
                    unsigned long long inj = launch ? q_inj : 0ull;
                    const unsigned lm = __ballot_sync(kFull, launch);
                    if (lm) {
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) inj += __shfl_xor_sync(kFull, inj, o);
                        if (lane == 0) atomicAdd(&s_cnt[LC_INJECTED_RAW], inj);
                    }
                }
                const unsigned flym = __ballot_sync(kFull, fly);
                if (fly) sts_u8(qR + nR + __popc(flym & lt_mask), slot);
                nR += __popc(flym);
                const unsigned unm = __ballot_sync(kFull, uninter);
                if (unm) {
                    if (uninter) sts_u8(qL + nL + __popc(unm & lt_mask), slot);
                    nL += __popc(unm);
                }
                __syncwarp();
            }
            if (nR == 0) break;                      // every slot of the pool is dead: the ticket is drained

            // =====================================================================================
            // CROSSING phase (Eq. 4): no RNG, no global memory, no branches in the crossing itself.
            // One crossing: d = r_c^2 - b^2 (negative: the surface is not reached, the lane stops with col
            // untouched); along-ray coordinate of the surface sn = +-sqrt(d); col -= rho^ (sn - s) (Eq. 4) is
            // committed together with the passage, and the lane stops if col < 0: the event lies col / rho^
            // before the surface (R7: an event exactly on a surface is a passage).
            // Flight state: along-ray coordinate s and impact parameter^2 b2 (units of R), remaining column col
            // (units of 1/kappa_ref) to the next event, shared-memory address pa of the candidate surface passage
            // (entry E); (pa - pa0) / 8 counts the passages since the package was taken from the pool.
            // =====================================================================================
            if (WT)
            {
                bool has = lane < nR;
                unsigned slot = 0, pa = tab0;
                // col: k_A-weighted column consumed (absorption clock, ends at cA0); colS: plain column (ends at cS0)
                float s = 0.f, b2 = 0.f, col = 1.f, colS = 0.f, cA0 = 0.f, cS0 = 0.f;
                if (has) {
                    slot = lds_u8(qR + (nR - 1 - lane));
                    const float4 a = lds_f4(aA + 16u * slot);
                    s = a.x; b2 = a.y; col = a.z; pa = __float_as_uint(a.w);
                    const float4 w4 = lds_f4(aW + 16u * slot);
                    colS = w4.x; cA0 = w4.y; cS0 = w4.z;
                }
                nR -= min(nR, 32);
                unsigned pa0 = pa;
                float4 E = lds_entry4(pa);
                bool alive = has;
                for (;;) {
                    const unsigned pb = pa;                      // the table is walked from here with constant offsets
#pragma unroll
                    for (int u = 0; u < kUnroll; u++) {
                        const float d = E.x - b2;
                        alive = alive && (d >= 0.f);
                        if (alive) {
                            // Eq. 4 for both clocks: absorption in k_A rho^, scattering in rho^ (its k_S sits in the draw)
                            const float sn = __int_as_float(__float_as_int(sqrt_ftz(d)) | (__float_as_int(E.y) & 0x80000000));
                            const float dl = sn - s;
                            col = fmaf(E.z, dl, col);
                            colS = fmaf(fabsf(E.y), dl, colS);
                            s = sn;
                            E = lds_entry4(pb + 16u * (u + 1));
                            pa = pb + 16u * (u + 1);
                        }
                        alive = alive && (col <= cA0) && (colS <= cS0);
                    }
                    {
                        // stopped short of a surface with both clocks still running (branch-free, as in the plain block).
                        // tang: the inner surface is not reached (tangent shell): head for the outer one instead, entry
                        // c -> entry 1 - c; the 1 - 2c entries skipped are no passages.  graze: outward, b2 > r^2 by
                        // rounding only.
                        const bool stop = !alive && (col <= cA0) && (colS <= cS0);
                        const bool tang = stop && (__float_as_int(E.y) < 0);
                        const bool graze = stop && !tang && (pa != pa_out);
                        const unsigned np = tang ? (2u * tab0 + 16u - pa) : pa;
                        pa0 += np - pa;
                        pa = np;
                        if (tang) E = lds_entry4(pa);
                        if (graze) b2 = E.x;
                        alive = alive || tang || graze;
                    }
                    const unsigned am = __ballot_sync(kFull, alive);
                    const int n_alive = __popc(am);
                    if (n_alive >= thr_hi) continue;
                    const bool leave = (nR == 0);
                    if (leave && n_alive >= thr_lo) continue;

                    // ---- stopped packages (all of them when leaving) go back to the pool and into their queues
                    const bool out = has && (leave || !alive);
                    int t = -1;
                    if (out) {
                        const bool isev = !alive && ((col > cA0) || (colS > cS0));   // a clock ran out
                        const unsigned n = ((pa - pa0) >> 4) - (isev ? 1u : 0u);
                        lc_cross += n;
                        if (TRACE) pT[2 * P + slot] += (int)n;
                        sts_f4(aA + 16u * slot, s, b2, col, __uint_as_float(pa));
                        sts_u32(aW + 16u * slot, __float_as_uint(colS));
                        t = alive ? QT_READY : QT_SRC;
                        if (isev) {
                            // the clock that ran out first along the step decides (R7: a tie is an absorption):
                            // distances back from the committed surface, (cA0 - col) / (k_A rho^) and (cS0 - colS) / rho^
                            const float4 Ep = lds_entry4(pa - 16u);
                            const float fA = col > cA0 ? (cA0 - col) / Ep.z : 3.0e38f;
                            const float fS = colS > cS0 ? (cS0 - colS) / fabsf(Ep.y) : 3.0e38f;
                            t = (fA <= fS) ? QT_ABS : QT_SCA;
                        }
                    }
                    {
                        // one store per leaving package: queue t at position (length of t) + (rank among the lanes of t)
                        const unsigned mA = __ballot_sync(kFull, t == QT_ABS), mS = __ballot_sync(kFull, t == QT_SCA);
                        const unsigned mL = __ballot_sync(kFull, t == QT_SRC), mR = __ballot_sync(kFull, t == QT_READY);
                        const unsigned mine = t == QT_ABS ? mA : t == QT_SCA ? mS : t == QT_SRC ? mL : mR;
                        const int base = t == QT_ABS ? nA : t == QT_SCA ? P + nS : t == QT_SRC ? 2 * P + nL : 3 * P + nR;
                        if (out) sts_u8(qA + base + __popc(mine & lt_mask), slot);
                        nA += __popc(mA); nS += __popc(mS); nL += __popc(mL); nR += __popc(mR);
                    }
                    __syncwarp();
                    if (leave) break;
                    // ---- idle lanes take the next ready packages
                    const unsigned fm = ~am;
                    const int r = __popc(fm & lt_mask);
                    const bool take = !alive && (r < nR);
                    if (take) {
                        slot = lds_u8(qR + (nR - 1 - r));
                        const float4 a = lds_f4(aA + 16u * slot);
                        s = a.x; b2 = a.y; col = a.z; pa = __float_as_uint(a.w);
                        const float4 w4 = lds_f4(aW + 16u * slot);
                        colS = w4.x; cA0 = w4.y; cS0 = w4.z;
                        pa0 = pa;
                        E = lds_entry4(pa);
                    } else if (!alive) {
                        col = 1.f; cA0 = 0.f;                    // idle lane: never flies, never looks stopped short
                    }
                    has = alive || take;
                    alive = has;
                    nR -= min(nR, __popc(fm));
                }
            }
            else
            {
                bool has = lane < nR;
                unsigned slot = 0, pa = tab0;
                float s = 0.f, b2 = 0.f, col = -1.f;
                if (has) {
                    slot = lds_u8(qR + (nR - 1 - lane));
                    const float4 a = lds_f4(aA + 16u * slot);
                    s = a.x; b2 = a.y; col = a.z; pa = __float_as_uint(a.w);
                }
                nR -= min(nR, 32);
                unsigned pa0 = pa;
                bool alive = has;
                // the along-ray coordinate is kept as a = +-s, positive along the direction of the entry the package
                // heads for (inward entries: a = -s), so that a new surface is a = sqrt(d) without a sign operation
                // and the signed density of the entry (negative: inward) does the rest
                float a = (pa <= tab0) ? -s : s;
                for (;;) {
                    // the table is walked from pb with constant offsets; the entries are read two steps ahead of their
                    // use and unconditionally (a lane that has stopped reads on harmlessly, at most 13 entries past its
                    // own, inside the block's shared memory), so that no crossing waits for a shared-memory load
                    const unsigned pb = pa;
                    float2 T0 = lds_entry(pb), T1 = lds_entry(pb + 8u);
#pragma unroll
                    for (int u = 0; u < kUnroll; u++) {
                        const float2 T2 = lds_entry(pb + 8u * (u + 2));
                        const float d = T0.x - b2;
                        alive = alive && (d >= 0.f);
                        if (alive) {
                            // col -= rho^ (sn - s) as (col + rho^ s) - rho^ sn with s = +-a, sn = +-sqrt(d), T0.y = +-rho^
                            const float t = fmaf(T0.y, a, col);
                            a = sqrt_ftz(d);
                            col = fmaf(-T0.y, a, t);
                            pa = pb + 8u * (u + 1);
                        }
                        alive = alive && (col >= 0.f);
                        T0 = T1; T1 = T2;
                    }
                    {
                        // stopped short of a surface with column left (branch-free: nearly every block has such lanes).
                        // tang: an inward entry (c <= 0) whose surface is not reached (tangent shell): head for the outer
                        // one instead, entry c -> entry 1 - c; the 1 - 2c entries skipped are no passages and the
                        // coordinate now runs along an outward entry.  graze: outward, b2 > r^2 by rounding only.
                        const bool stop = !alive && (col >= 0.f);
                        const bool tang = stop && (pa <= tab0);
                        const bool graze = stop && (pa > tab0) && (pa != pa_out);
                        const unsigned np = tang ? (2u * tab0 + 8u - pa) : pa;
                        pa0 += np - pa;
                        pa = np;
                        a = tang ? -a : a;
                        if (graze) b2 = lds_entry(pa).x;
                        alive = alive || tang || graze;
                    }
                    const unsigned am = __ballot_sync(kFull, alive);
                    const int n_alive = __popc(am);
                    if (n_alive >= thr_hi) continue;
                    const bool leave = (nR == 0);
                    if (leave && n_alive >= thr_lo) continue;

                    // ---- stopped packages (all of them when leaving) go back to the pool and into their queues
                    const bool out = has && (leave || !alive);
                    int t = -1;
                    if (out) {
                        const unsigned kf = lds_u32(aB + 16u * slot + 12u);
                        const bool isev = !alive && (col < 0.f);         // the column ran out: scattering or absorption
                        const unsigned n = ((pa - pa0) >> 3) - (isev ? 1u : 0u);
                        lc_cross += n;
                        if (TRACE) pT[2 * P + slot] += (int)n;
                        // signed coordinate: a runs along the entry ahead (flying) or the one just committed (event)
                        s = ((alive ? pa : pa - 8u) <= tab0) ? -a : a;
                        sts_f4(aA + 16u * slot, s, b2, col, __uint_as_float(pa));
                        // stopped on the sentinel: left the model
                        t = alive ? QT_READY : (isev ? ((kf & KF_EVABS) ? QT_ABS : QT_SCA) : QT_SRC);
                    }
                    {
                        // one store per leaving package: queue t at position (length of t) + (rank among the lanes of t)
                        const unsigned mA = __ballot_sync(kFull, t == QT_ABS), mS = __ballot_sync(kFull, t == QT_SCA);
                        const unsigned mL = __ballot_sync(kFull, t == QT_SRC), mR = leave ? am : 0u;   // flying lanes leave only at the end
                        const unsigned mine = t == QT_ABS ? mA : t == QT_SCA ? mS : t == QT_SRC ? mL : mR;
                        const int base = t == QT_ABS ? nA : t == QT_SCA ? P + nS : t == QT_SRC ? 2 * P + nL : 3 * P + nR;
                        if (out) sts_u8(qA + base + __popc(mine & lt_mask), slot);
                        nA += __popc(mA); nS += __popc(mS); nL += __popc(mL); nR += __popc(mR);
                    }
                    __syncwarp();
                    if (leave) break;
                    // ---- idle lanes take the next ready packages
                    const unsigned fm = ~am;
                    const int r = __popc(fm & lt_mask);
                    const bool take = !alive && (r < nR);
                    if (take) {
                        slot = lds_u8(qR + (nR - 1 - r));
                        const float4 a4 = lds_f4(aA + 16u * slot);
                        s = a4.x; b2 = a4.y; col = a4.z; pa = __float_as_uint(a4.w);
                        a = (pa <= tab0) ? -s : s;
                        pa0 = pa;
                    } else if (!alive) {
                        col = -1.f;                              // idle lane: never flies, never looks stopped short
                    }
                    has = alive || take;
                    alive = has;
                    nR -= min(nR, __popc(fm));
                }
            }
            // counters: flush before a 32-bit count can wrap
            if (__any_sync(kFull, ((lc_cross | lc_ffi | wc_pkg | wc_sca | wc_abs | wc_esc) >> 30) != 0u)) {
                atomicAdd(&s_cnt[LC_CROSSINGS], (unsigned long long)lc_cross);
                if (lc_ffi) atomicAdd(&s_cnt[LC_FFI_CROSSINGS], (unsigned long long)lc_ffi);
                if (lane == 0) {
                    atomicAdd(&s_cnt[LC_PACKAGES], (unsigned long long)wc_pkg);
                    atomicAdd(&s_cnt[LC_SCATTERINGS], (unsigned long long)wc_sca);
                    atomicAdd(&s_cnt[LC_ABSORPTIONS], (unsigned long long)wc_abs);
                    atomicAdd(&s_cnt[LC_ESCAPED], (unsigned long long)wc_esc);
                    if (R.uniform_q) atomicAdd(&s_cnt[LC_INJECTED_RAW], q_uni * (unsigned long long)wc_pkg);
                }
                lc_cross = lc_ffi = wc_pkg = wc_sca = wc_abs = wc_esc = 0u;
            }
        }
        // ---------------- per-ticket flush of the warp's counts (identical quanta: injected raw units = launches x quantum)
        {
            unsigned long long c = lc_cross, f = lc_ffi;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { c += __shfl_xor_sync(kFull, c, o); f += __shfl_xor_sync(kFull, f, o); }
            if (lane == 0) {
                atomicAdd(&s_cnt[LC_CROSSINGS], c);
                if (f) atomicAdd(&s_cnt[LC_FFI_CROSSINGS], f);
                atomicAdd(&s_cnt[LC_PACKAGES], (unsigned long long)wc_pkg);
                atomicAdd(&s_cnt[LC_SCATTERINGS], (unsigned long long)wc_sca);
                atomicAdd(&s_cnt[LC_ABSORPTIONS], (unsigned long long)wc_abs);
                atomicAdd(&s_cnt[LC_ESCAPED], (unsigned long long)wc_esc);
                if (R.uniform_q) atomicAdd(&s_cnt[LC_INJECTED_RAW], q_uni * (unsigned long long)wc_pkg);
            }
            lc_cross = lc_ffi = wc_pkg = wc_sca = wc_abs = wc_esc = 0u;
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
