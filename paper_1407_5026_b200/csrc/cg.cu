// cg.cu — libcg.so: parallel-rejection kinetic Monte Carlo of the 2D Coulomb glass
// (Ferrero, Kolton, Palassini, arXiv 1407.5026) for NVIDIA B200 (sm_100a).
//
// The ABI is declared and documented in include/cg.h.  DESIGN.md explains the
// kernel design; the short version:
//   * one persistent cooperative kernel runs the whole propose -> select ->
//     apply -> update loop, one CTA per SM; in each CTA 14 worker
//     warps test proposals and update eps, a control warp does the exchange and the
//     bookkeeping, a service warp publishes finished slab updates;
//   * the grid exchange is one-way most of the time: slots are scanned in label
//     order and the scan stops at the first accepting CTA, so the CTA that holds
//     the start of the window never waits for the others;
//   * every thread owns the attempts a = g (mod P), keeps its proposal decoded and,
//     while theta_ij = 1, follows the two local energies it needs in registers by
//     adding every executed hop's term itself (the same rounded adds as the update);
//   * each CTA keeps its eps slab in registers and writes it through to a ring of
//     buffers; readers only touch a buffer that every CTA has published and add the
//     terms of the (at most CG_DEPTH) newer hops in hop order, so no reader ever
//     waits for a writer and every value is bit-identical to the serial algorithm;
//   * occupations live as a bitmap in every CTA's shared memory, next to the live
//     part of the tower and its guide table; 1/r comes from an
//     unfolded table in L2 indexed with one subtraction and one mask.
// Nothing in this file is shared with oracle/ (the CPU reference).
#include "cg.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

typedef unsigned long long u64;
typedef unsigned int u32;

#define CG_NONE 0xFFFFFFFFu
#define CG_FULL 0xFFFFFFFFu
#define CG_MAX_CTAS 1024

// ------------------------------------------------------------------ device --

#ifndef CG_DEPTH
#define CG_DEPTH 4          // pending hops: proposals read eps_{h-DEPTH} and add the newer hops' terms themselves
#endif
#define CG_RING (2 * CG_DEPTH + 1)   // eps buffers: eps_{h+1-2 DEPTH} .. eps_{h+1} can be live at the same time
#define CG_SRING 16         // exchange slots per CTA: a CTA posts up to DEPTH exchanges ahead of the slowest reader
#define CG_PUB_U64 32       // offset of a CTA's publication word in its slot block (u64 units)
#define CG_SLOT_U64 64      // one block per CTA, 512-byte stride: the slot ring in the first half, the pub word after it
#define CG_GUIDE 352        // tower guide: (43 + 1) binades x 8 sub-buckets of t = 2^43 - m

struct CgCtl {              // device-resident control block (one per sim)
    u64 attempts;           // attempts consumed = next unused attempt index
    u64 hops;               // executed hops
    u64 iterations;         // PR iterations
    u64 proposals;          // proposals evaluated (M per iteration)
    long long dP;           // sum of dx over executed hops
    u32 cur;                // eps buffer that holds the complete current state
    u32 bad_hops;           // scripted hops that violated theta_ij
    u64 epoch;              // next exchange epoch; never reset, so stale slots can never match
    u64 log_base;           // hop count at which the hop log was enabled
    u64 cyc_total, cyc_wait, cyc_update, cyc_propose;
    u64 pub_base;           // publication sequence number of the last hop of the previous launch: CTA c
                            // stores pub_base + h into its pub word once its slab of hop h of a launch is
                            // written (never reset, so stale words of other launch shapes are always smaller)
    u64 log_a0;             // attempts consumed when the hop log was enabled (observables: m of the first logged hop)
    u64 pub_pad[2];
};

struct CgParams {           // kernel parameter block
    double* eps[CG_RING];   // ring of local-energy buffers, N each (see "pending hops" below)
    const double* tf;       // unfolded table 1/r, L rows of pitch 2L (see site_code)
    const double* tq;       // quarter table 1/r, (L/2+1) x (L/2+1), indexed by the folded offsets
    u32* nbits;             // occupations, bit s of word s/32
    const u64* cdfi;        // live tower as integer thresholds: u_d < cdf_k  <=>  m < cdfi_k
    const double* invr_k;   // 1/r of displacement k (live part)
    const double* fld_k;    // E * dx of displacement k
    const int* disp;        // (dy << 16) | (dx & 0xffff)
    const u32* guide;       // tower guide: klo | khi << 16 per bucket
    u64* slots;             // exchange slots, CG_SLOT_U64 per CTA
    CgCtl* ctl;
    u64* log_a; u32* log_i; u32* log_j; u64 log_cap;
    int L, lgL, pitch, Klive;
    u32 N, M;
    u32 PL;                 // CACHED: threads per CTA that own attempts
    u32 seed_lo, seed_hi;
    double T, E;
    float inv_T;            // (float)(1/T), pre-test of the Metropolis factor only
    u64 n_hops;
    u64* trace;             // optional segment timers (cg_set_trace), 64 words per CTA
    u32 trace_iters;
};

// Philox4x32-10 (Salmon et al., SC'11): counter (c0..c3), key (k0,k1).
__device__ __forceinline__ void philox4x32_10(u32 c0, u32 c1, u32 c2, u32 c3, u32 k0, u32 k1,
                                              u32& o0, u32& o1, u32& o2, u32& o3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const u32 hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const u32 hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const u32 t0 = hi1 ^ c1 ^ k0, t2 = hi0 ^ c3 ^ k1;
        c0 = t0; c1 = lo1; c2 = t2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

__device__ __forceinline__ double ld_cg(const double* p) { return __ldcg(p); }

__device__ __forceinline__ void slot_store(u64* p, u64 a, u64 b)
{
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void slot_load(const u64* p, u64& a, u64& b)
{
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ u64 ld_relaxed_u64(const u64* p)
{
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(u64* p, u64 v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ u64 global_ns()
{
    u64 t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void fence_acquire_gpu() { asm volatile("fence.acquire.gpu;" ::: "memory"); }
// named barriers 1 .. CG_DEPTH (cyclic in the hop number): the warps that wrote eps arrive, the
// service warp waits for them; barrier 0 with an explicit count synchronises the worker warps only
#define CG_BARN(OP) switch (k) { \
        case 0: asm volatile(OP " 1, %0;" ::"r"(n) : "memory"); break; \
        case 1: asm volatile(OP " 2, %0;" ::"r"(n) : "memory"); break; \
        case 2: asm volatile(OP " 3, %0;" ::"r"(n) : "memory"); break; \
        case 3: asm volatile(OP " 4, %0;" ::"r"(n) : "memory"); break; \
        case 4: asm volatile(OP " 6, %0;" ::"r"(n) : "memory"); break; \
        case 5: asm volatile(OP " 7, %0;" ::"r"(n) : "memory"); break; \
        case 6: asm volatile(OP " 8, %0;" ::"r"(n) : "memory"); break; \
        default: asm volatile(OP " 9, %0;" ::"r"(n) : "memory"); break; }
__device__ __forceinline__ void barN_arrive(u32 k, int n) { CG_BARN("bar.arrive") }   // k < CG_DEPTH <= 8
__device__ __forceinline__ void barN_sync(u32 k, int n) { CG_BARN("bar.sync") }
__device__ __forceinline__ void barX_sync(int n) { asm volatile("bar.sync 0, %0;" ::"r"(n) : "memory"); }
__device__ __forceinline__ void barX_arrive(int n) { asm volatile("bar.arrive 0, %0;" ::"r"(n) : "memory"); }
// barrier 5: second CTA barrier of an iteration; the control warp only arrives
__device__ __forceinline__ void barB_sync(int n) { asm volatile("bar.sync 5, %0;" ::"r"(n) : "memory"); }
__device__ __forceinline__ void barB_arrive(int n) { asm volatile("bar.arrive 5, %0;" ::"r"(n) : "memory"); }

// ---- the unfolded 1/r table ------------------------------------------------------------
// tf[dy * 2L + dx] = 1/r of the offset (dy, dx) under minimum image, dy in [0, L),
// dx in [0, L] (dx = L repeats dx = 0, so the pair (dx, dx+1) never wraps); 0 at the origin.
// A site s = y L + x is coded as c(s) = y 2L + x; with bit L (the spare bit between the fields) set
// in the minuend, ONE subtraction and ONE mask give both periodic differences:
//   ((c(s) | L) - c(t)) & mask  =  ((y_s - y_t) mod L) 2L + ((x_s - x_t) mod L).
__device__ __forceinline__ u32 site_code(u32 s, int L) { return s + (s & ~(u32)(L - 1)); }

// Step 3b of the mixed PR algorithm: what hop i->j adds to eps at the site coded sc
// (spare bit set): 1/r_lj - 1/r_li (difference first, then ONE add by the caller).
__device__ __forceinline__ double hop_term(const double* __restrict__ tf, u32 mask, u32 sc, u32 ci, u32 cj)
{
    return __dsub_rn(__ldg(tf + ((sc - cj) & mask)), __ldg(tf + ((sc - ci) & mask)));
}

// eps slab of one CTA: sites [2 pr0, 2 pr1).  With RP > 0 warp w keeps the blocks of 64 consecutive
// sites number w, w + TW/32, ... (RP of them) in registers across hops - lane l holds sites l and
// 32 + l of a block, so that every load and store of the warp covers 256 contiguous bytes (the L1
// wavefront rate, not L2 bandwidth, bounds this kernel) - and writes every new value through to global
// memory for the other CTAs' gathers; with RP == 0 the slab streams src -> dst.
// issue() starts the table gathers of a hop, finish() adds and stores: the caller puts independent
// work between the two.
template <int TW, int RP>
struct Slab {
    static constexpr int R = RP > 0 ? RP : 1;
    double ea[R], eb[R];
    double ja[R], ia[R], jb[R], ib[R];
    u32 sca[R], scb[R];                  // coded sites (spare bit set); 0 marks a site outside the slab
    u32 hci, hcj;
    u32 tix;                             // index of this thread among the TW threads that hold the slab

    __device__ __forceinline__ u32 site_a(u32 pr0, int k) const
    {
        return 2u * (pr0 + (u32)k * TW + (tix & ~31u)) + (tix & 31u);
    }

    __device__ __forceinline__ void load(const double* src, u32 pr0, u32 pr1, int L, u32 t)
    {
        tix = t;
#pragma unroll
        for (int k = 0; k < RP; ++k) {
            const u32 sa = site_a(pr0, k), sb = sa + 32u;
            sca[k] = sa < 2u * pr1 ? site_code(sa, L) | (u32)L : 0u;
            scb[k] = sb < 2u * pr1 ? site_code(sb, L) | (u32)L : 0u;
            if (sca[k]) ea[k] = __ldcg(src + sa);
            if (scb[k]) eb[k] = __ldcg(src + sb);
        }
    }

    __device__ __forceinline__ void issue(const double* __restrict__ tf, u32 mask, u32 pr0, u32 pr1, u32 ci, u32 cj)
    {
        hci = ci; hcj = cj;
#pragma unroll
        for (int k = 0; k < RP; ++k) {
            if (sca[k]) { ja[k] = __ldg(tf + ((sca[k] - cj) & mask)); ia[k] = __ldg(tf + ((sca[k] - ci) & mask)); }
            if (scb[k]) { jb[k] = __ldg(tf + ((scb[k] - cj) & mask)); ib[k] = __ldg(tf + ((scb[k] - ci) & mask)); }
        }
    }

    // dst = eps + (1/r_lj - 1/r_li) for every site l of the slab
    __device__ __forceinline__ void finish(const double* __restrict__ tf, u32 mask, int L, const double* src,
                                           double* dst, u32 pr0, u32 pr1)
    {
        if (RP > 0) {
#pragma unroll
            for (int k = 0; k < RP; ++k) {
                const u32 sa = site_a(pr0, k);
                if (sca[k]) { ea[k] = __dadd_rn(ea[k], __dsub_rn(ja[k], ia[k])); __stcg(dst + sa, ea[k]); }
                if (scb[k]) { eb[k] = __dadd_rn(eb[k], __dsub_rn(jb[k], ib[k])); __stcg(dst + sa + 32u, eb[k]); }
            }
        } else {
            for (u32 s = 2u * pr0 + tix; s < 2u * pr1; s += TW) {
                const u32 c = site_code(s, L) | (u32)L;
                const double v = __ldcg(src + s);
                const double tj = __ldg(tf + ((c - hcj) & mask)), ti = __ldg(tf + ((c - hci) & mask));
                __stcg(dst + s, __dadd_rn(v, __dsub_rn(tj, ti)));
            }
        }
    }
};

struct Prop {               // one decoded attempt (a pure function of seed and attempt index)
    u32 i, j, k;            // sites and tower index
    u32 uh, ul;             // the 53 acceptance bits: u_a = (uh 2^32 + ul) 2^-53, uh < 2^21
};

struct Tables {             // shared-memory views
    const u64* cdfi; const double* invr; const double* fld; const int* disp; const u32* guide;
};

// Tower sampling: smallest k with u_d < cdf_k, u_d = m 2^-43, as the equivalent integer
// test m < cdfi_k; the guide brackets k from the leading bits of t = 2^43 - m (the tail of the tower is
// geometric, so a binade of t holds only a few k).
__device__ __forceinline__ u32 tower_search(const Tables& t, u64 m)
{
    const u64 tt = (1ull << 43) - m;
    const int e = 63 - __clzll((long long)tt);
    const u32 mant = (e >= 3 ? (u32)(tt >> (e - 3)) : (u32)(tt << (3 - e))) & 7u;
    const u32 g = t.guide[e * 8 + (int)mant];
    u32 lo = g & 0xFFFFu, hi = g >> 16;
    while (lo < hi) {
        const u32 mid = (lo + hi) >> 1;
        if (m < t.cdfi[mid]) hi = mid; else lo = mid + 1;
    }
    return lo;
}

__device__ __forceinline__ u32 hop_target(const Tables& t, u32 i, u32 k, int L, int lg)
{
    const int d = t.disp[k];
    const int dy = d >> 16, dx = (int)(short)(d & 0xFFFF);
    const int yj = ((int)(i >> lg) + dy) & (L - 1), xj = ((int)(i & (L - 1)) + dx) & (L - 1);
    return ((u32)yj << lg) | (u32)xj;
}

// Attempt a -> proposal (reading G9): one Philox block, i = (w0 N) >> 32,
// displacement from 43 bits, acceptance uniform from the remaining 53.
__device__ __forceinline__ Prop decode_attempt(const Tables& t, const CgParams& p, u64 a)
{
    u32 w0, w1, w2, w3;
    philox4x32_10((u32)a, (u32)(a >> 32), 0u, 0u, p.seed_lo, p.seed_hi, w0, w1, w2, w3);
    Prop r;
    r.i = __umulhi(w0, p.N);
    r.k = tower_search(t, ((u64)w1 << 11) | (u64)(w2 >> 21));
    r.j = hop_target(t, r.i, r.k, p.L, p.lgL);
    r.uh = w2 & 0x1FFFFFu; r.ul = w3;
    return r;
}

// Eq.(2): for dE > 0 accept iff u_a < exp(-dE/T).  A float estimate with a 2^-10 guard
// band decides all but near-ties; those take the double-precision path, so the decision is always
// that of the double comparison.
__device__ __forceinline__ bool metropolis(double dE, u32 uh, u32 ul, double T, float inv_T)
{
    if (dE <= 0.0) return true;
    const u32 top = (uh << 11) | (ul >> 21);                       // top 32 of the 53 bits
    const float lo = (float)top * 2.3283064365386963e-10f;         // u_a in [lo, lo + 2^-32)
    const float xf = (float)(-dE) * inv_T;
    const float pf = __expf(xf);
    if (lo > pf * 1.0009765625f) return false;
    if (xf > -60.f && lo + 4.6566128730773926e-10f < pf * 0.9990234375f) return true;
    const double ua = (double)(((u64)uh << 32) | (u64)ul) * (1.0 / 9007199254740992.0);
    return ua < exp(__ddiv_rn(-dE, T));
}

#define BIT(sn, s) (((sn)[(s) >> 5] >> ((s) & 31)) & 1u)

#ifdef CG_TRACE
// segment timers of thread 0 (SM cycles), summed over the launch, separately for iterations in which
// this CTA held the start of the window (class 0) or not (class 1): p.trace[b*32 + class*16 + segment]
#define CLS_ (kb == 0 ? 0 : kb == 1 ? 32 : kb == nb - 1 ? 48 : 16)
#define TRACE(ev, extra) do { if (lane == 0) { const long long now_ = clock64(); \
    s_seg[CLS_ + (ev)] += (u64)(now_ - t_prev); t_prev = now_; } } while (0)
#elif defined(CG_TRACE_W)
#define TRACE(ev, extra) do { const long long now_ = clock64(); cw[ev] += (u64)(now_ - cprev); cprev = now_; } while (0)
#else
#define TRACE(ev, extra) do { } while (0)
#endif
#ifdef CG_TRACE_T
// Time line: absolute SM clocks of 64 consecutive iterations (2000..2063 of a launch) of CTAs 0..31,
// p.trace[((it - 2000) * 32 + b) * 32 + k]: k < 10 control warp (loop top, publication check done, early look
// done, arrival at [A], CTA minimum, posted, scan done, before [B], arrived at [B], end), 10 scan position,
// 11 attempts consumed; 16 + k worker warp 0 and 24 + k last worker warp (proposals known, tested, warp
// minimum stored, [A] done, slab update done, [B] done, descriptor read, loop top).
__device__ __forceinline__ u64 clk_now() { u64 t; asm volatile("mov.u64 %0, %%clock64;" : "=l"(t) :: "memory"); return t; }
#define TS_CTL(k) do { if (lane == 0 && p.trace && b < 32u && it_local - 2000u < 64u) \
    p.trace[((it_local - 2000u) * 32u + b) * 32u + (k)] = clk_now(); } while (0)
#define TS_WRK(k) do { if (lane == 0 && (warp == 0 || warp == NWK - 1) && p.trace && b < 32u && itw - 2000u < 64u) \
    p.trace[((itw - 2000u) * 32u + b) * 32u + 16u + (warp ? 8u : 0u) + (k)] = clk_now(); } while (0)
#else
#define TS_CTL(k) do { } while (0)
#define TS_WRK(k) do { } while (0)
#endif

// What warp 0 tells the other warps of its CTA about an exchange (written before the second barrier).
struct Desc {
    u32 used;               // attempts consumed: q + 1, or M when the whole window was rejected
    u32 hop;                // 1: a hop was executed
    u32 ci, cj;             // its coded sites (site_code)
    u32 ahead;              // 1: another CTA holds the start of the next window (time to decode ahead)
    u32 pad[3];
};
struct Pend {               // pending hops, for threads that start to follow a pair of sites
    u32 npend, rbuf, first, pad;   // buffer rbuf + the npend hops c[(first + k) % CG_DEPTH], k = 0.. (oldest first)
    u32 c[CG_DEPTH][2];     // coded sites (i, j) of the last CG_DEPTH executed hops, hop number h at (h - 1) % CG_DEPTH
};
static_assert(CG_DEPTH <= 8 && CG_DEPTH < CG_SRING, "named barriers, slot ring");

// The persistent kernel: steps 1, 2, 3a-3c of the mixed PR algorithm.
// CACHED: thread g of the grid owns the attempts a = g (mod P), P = gridDim.x * PL >= M, keeps its
// current and its next proposal decoded in registers (a proposal is a pure function of the seed and
// the attempt index) and, while theta_ij = 1, also the two local energies it needs, to which it adds
// the term of every executed hop itself; an iteration then only re-tests the proposal on the current
// state.  Otherwise CTA b evaluates labels [b per, (b+1) per) from scratch.
// Warp 0 of every CTA does the exchange and all bookkeeping; the other worker warps only test their
// proposals and update their part of the eps slab, and learn the outcome from a small descriptor.
// Written as a device function of (parameters, CTA index, CTA count) so that one launch can also hold
// several sims side by side (cg_pr_persistent_many): nothing in it looks at blockIdx or gridDim, and all
// synchronisation between CTAs goes through the sim's own slots and publication words.
template <int THREADS, int RP, bool CACHED>
__device__ __forceinline__ void pr_persistent_body(const CgParams& p, const u32 b, const u32 nb)
{
    constexpr int TW = THREADS - 64;      // worker threads; then the control warp and the service warp
    constexpr int NWK = TW / 32;          // worker warps = index of the control warp
    constexpr int TB = TW + 32;           // threads at the CTA barriers of an iteration (workers + control)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int KL = p.Klive;
    u64* s_cdfi = reinterpret_cast<u64*>(smem_raw);
    double* s_invr = reinterpret_cast<double*>(s_cdfi + KL);
    double* s_fld = s_invr + KL;
    int* s_disp = reinterpret_cast<int*>(s_fld + KL);
    u32* s_guide = reinterpret_cast<u32*>(s_disp + KL);
    u32* s_n = s_guide + CG_GUIDE;
    __shared__ u32 s_key;                 // lowest accepting (label << 5 | warp) of the CTA in this iteration
    __shared__ u64 s_wpay[32];            // (i, j) of each warp's lowest accepting label
    __shared__ u64 s_verified;            // newest publication sequence number seen from ALL CTAs (service warp)
    __shared__ __align__(16) Desc s_desc;
    __shared__ __align__(16) Pend s_pend;
    const Tables tb = {s_cdfi, s_invr, s_fld, s_disp, s_guide};
#ifdef CG_TRACE
    __shared__ u64 s_seg[64];
    if (threadIdx.x < 64) s_seg[threadIdx.x] = 0;
    long long t_prev = 0;
#endif

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int L = p.L, lg = p.lgL;
    const u32 N = p.N, M = p.M;
    const u32 mask = ((u32)(L - 1) << (lg + 1)) | (u32)(L - 1);
    const double* __restrict__ tf = p.tf;

    for (int k = tid; k < KL; k += THREADS) {
        s_cdfi[k] = p.cdfi[k]; s_invr[k] = p.invr_k[k]; s_fld[k] = p.fld_k[k]; s_disp[k] = p.disp[k];
    }
    for (int k = tid; k < CG_GUIDE; k += THREADS) s_guide[k] = p.guide[k];
    for (u32 w = tid; w < (N + 31) / 32; w += THREADS) s_n[w] = p.nbits[w];
    if (tid == 0) {
        s_key = CG_NONE;
        s_verified = p.ctl->pub_base;
        s_pend.npend = 0; s_pend.rbuf = p.ctl->cur; s_pend.first = 0;
    }

    const u64 a_start = p.ctl->attempts, pub_base = p.ctl->pub_base;
    u64 hl = 0;                           // hops executed in this launch
    u32 wbuf = p.ctl->cur;                // buffer of the ring that holds the newest eps
    bool upd = false;                     // slab update issued, not yet finished
    bool newhop = false;                  // the previous iteration executed a hop ...
    u32 hci = 0, hcj = 0;                 // ... with these coded sites
    bool ahead = false;                   // another CTA holds the start of the window
    const long long t_begin = clock64();

    // labels: CTA-blocked (scan order = CTA order) or, CACHED, cyclic in the global thread index
    const u32 per = CACHED ? p.PL : (M + nb - 1) / nb;
    const u32 lab0 = min(M, b * per), lab1 = min(M, lab0 + per);
    const u32 P = nb * per;               // CACHED: attempts a = g (mod P) belong to thread g
    u32 c_first = 0, t0r = 0;             // CACHED: CTA at scan position 0 and the offset of a0 in it
    if (CACHED) { const u32 g0 = (u32)(a_start % P); c_first = g0 / per; t0r = g0 - c_first * per; }
    const bool has_label = CACHED && (u32)tid < per;
    __syncthreads();
    if (warp == NWK + 1) {
        // service warp: once per executed hop, wait until every worker has stored its part of the
        // slab (named barrier), fence those stores and bump the publication counter - off the
        // workers' critical path.  Workers run at most CG_DEPTH hops ahead of it (the exchange of hop
        // h+DEPTH waits for the publication of hop h by every CTA, this one included), hence as many
        // barriers.
        // After publishing it looks at every CTA's publication word once and leaves the newest hop that
        // ALL of them have published in shared memory: the control warp, which must know that before it
        // lets a hop through, then rarely has to look itself.
        if (nb > 1)
            for (u64 h = 0; h < p.n_hops; ++h) {
                barN_sync((u32)(h % CG_DEPTH), TB);
                if (lane == 0) st_release_u64(p.slots + (size_t)b * CG_SLOT_U64 + CG_PUB_U64, pub_base + h + 1);
                u64 vmin = ~0ull;
                for (u32 c0 = lane; c0 < nb; c0 += 32 * 8) {            // eight independent loads in flight
                    u64 v[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const u32 c = c0 + 32 * k;
                        v[k] = c < nb ? ld_relaxed_u64(p.slots + (size_t)c * CG_SLOT_U64 + CG_PUB_U64) : ~0ull;
                    }
#pragma unroll
                    for (int k = 0; k < 8; ++k) vmin = min(vmin, v[k]);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) vmin = min(vmin, __shfl_xor_sync(CG_FULL, vmin, o));
                fence_acquire_gpu();
                if (lane == 0 && vmin > pub_base) *(volatile u64*)&s_verified = vmin;    // stale words are smaller
            }
        return;
    }
    // CACHED per-thread state: label of my attempt relative to the window start, the decoded proposal
    // and what its test needs; the attempt after it, decoded ahead when there is idle time
    u32 lab = CG_NONE;
    u64 a_cur = 0;
    u32 ci_ = 0, cj_ = 0, sci = 0, scj = 0, cuh = 0, cul = 0;
    double c_invr = 0, c_fld = 0, ei = 0, ej = 0;
    bool tracked = false;                 // ei, ej hold the current local energies of my two sites
    Prop nxt = {0, 0, 0, 0, 0};
    bool nxt_valid = false;
    auto take = [&](const Prop& q) {
        ci_ = q.i; cj_ = q.j; cuh = q.uh; cul = q.ul;
        sci = site_code(q.i, L) | (u32)L; scj = site_code(q.j, L) | (u32)L;
        c_invr = s_invr[q.k]; c_fld = s_fld[q.k];
        tracked = false;
    };
    if (has_label) {
        const u32 g = b * per + (u32)tid, g0 = c_first * per + t0r;
        lab = g >= g0 ? g - g0 : g + P - g0;
        a_cur = a_start + lab;
        take(decode_attempt(tb, p, a_cur));
    }
    ahead = CACHED && c_first != b;

    const u32 pairs = N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    u64* const my_slot = p.slots + (size_t)b * CG_SLOT_U64;

    if (warp == NWK) {
        // ------------------------------------------------------------------ control warp ----
        // Exchange and bookkeeping of the CTA; it holds no labels and no eps.
        const u64 log_base = p.ctl->log_base, hops_start = p.ctl->hops;
        const u32 e_start = (u32)p.ctl->epoch;
        u64 used_sum = 0;                 // attempts consumed in this launch
        long long dP = 0;
        u32 it_local = 0;                 // PR iterations of this launch
        // Pending hops.  eps lives in a ring of CG_RING buffers: hop h writes eps_h (each CTA its own
        // slab) into the buffer after the one hop h-1 wrote.  Nobody reads buffers that other CTAs may
        // still be writing: a proposal that starts to follow a pair of sites reads eps_v, v = the newest
        // hop every CTA has published (buffer rbuf; v >= h - DEPTH by the publication check), and adds
        // the terms 1/r_lj - 1/r_li of the hops v+1 .. h itself, in hop order - the same single rounded
        // adds the update performs, so the values are bit-identical whatever v is.  A CTA writes
        // eps_{h'} only when every CTA has published hop h' - DEPTH; a reader at hop h has published
        // at most h, so h' <= h + DEPTH while it reads v >= h - DEPTH: with 2 DEPTH + 1 buffers a
        // buffer is never written while read.
        const u32 cur0 = wbuf;            // buffer that holds eps at the start of this launch
        // CTA c has published hop number h of this launch once its pub word is >= pub_base + h
        u64 need_pub = 0;                 // hop hl - DEPTH + 1: readers never reach back further than DEPTH hops
        u64 ver = pub_base;               // newest publication seen from ALL CTAs
#ifdef CG_TRACE_W
        u64 cw[16] = {}; long long cprev = clock64();
#endif
        while (hl < p.n_hops) {
            const u32 e32 = e_start + it_local;
            const u32 kb = b >= c_first ? b - c_first : b + nb - c_first;    // my scan position
            TS_CTL(0);
#ifdef CG_TRACE
            if (lane == 0) { if (t_prev == 0) t_prev = clock64(); s_seg[CLS_ + 15] += 1; }
#endif
            // Hop hl - DEPTH + 1 must be complete on every CTA before the workers of this CTA are let into the
            // next iteration (readers reach back at most DEPTH hops): one publication word per CTA, each in its
            // own L2 slice.  This warp is idle while the workers test their proposals, so the check is free.
            if (nb > 1) ver = max(ver, *(volatile u64*)&s_verified);
            if (nb > 1 && ver < need_pub) {                             // rarely: the service warp has usually seen it
                for (;;) {
                    bool ok = true;
                    for (u32 c0 = lane; c0 < nb; c0 += 32 * 8) {        // eight independent loads in flight
                        u64 v[8];
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const u32 c = c0 + 32 * k;
                            v[k] = c < nb ? ld_relaxed_u64(p.slots + (size_t)c * CG_SLOT_U64 + CG_PUB_U64) : ~0ull;
                        }
#pragma unroll
                        for (int k = 0; k < 8; ++k) ok = ok && v[k] >= need_pub;
                    }
#ifdef CG_TRACE
                    if (lane == 0) s_seg[CLS_ + 8] += 1;      // passes of the publication check
#endif
                    if (__all_sync(CG_FULL, ok)) break;
                }
                fence_acquire_gpu();
                ver = need_pub;
            }
            TRACE(6, 0);
            TS_CTL(1);
            // A CTA that does not hold the start of the window usually runs behind the one that does: the
            // winner of this exchange may already be posted.  One look at the first two scan positions
            // before the barrier takes that round trip off the path between the two barriers.
            const u32 tail0 = CACHED ? per - t0r : CG_NONE;            // position 0: labels >= tail0 are tail labels
            const u32 ring = (e32 & (CG_SRING - 1u)) * 2u;
            const u32 e16 = e32 & 0xFFFFu;
            u32 eq = CG_NONE; u64 ewp = 0;
            if (nb > 1 && kb != 0) {
                const bool mine = lane < 2 && (u32)lane < kb;
                u32 c = c_first + lane; if (c >= nb) c -= nb;
                u32 l = CG_NONE; u64 q0 = 0, q1 = 0; bool ready = false;
                if (mine) {
                    slot_load(p.slots + (size_t)c * CG_SLOT_U64 + ring, q0, q1);
                    ready = (u32)(q0 >> 32) == e32 && (u32)(q1 >> 48) == e16;
                    l = ready ? (u32)q0 : CG_NONE;
                    if (CACHED && lane == 0 && l != CG_NONE && l >= tail0) l = CG_NONE;    // tail labels never win early
                }
                const u32 racc = __ballot_sync(CG_FULL, mine && ready && l != CG_NONE);
                const u32 rnot = __ballot_sync(CG_FULL, mine && !ready);
                const int fa = racc ? __ffs(racc) - 1 : 32, fn = rnot ? __ffs(rnot) - 1 : 32;
                if (fa < fn) {
                    eq = __shfl_sync(CG_FULL, l, fa);
                    ewp = __shfl_sync(CG_FULL, q1, fa);
                    ewp = ((ewp >> 24) & 0xFFFFFFull) << 32 | (ewp & 0xFFFFFFull);
                }
            }
            TRACE(7, 0);
#ifdef CG_TRACE_W
            cw[15] += 1; if (eq != CG_NONE) cw[14] += 1; if (kb == 0) cw[13] += 1;
#endif
            TS_CTL(2);
            barX_sync(TB);                // [A] the workers have tested their proposals
            TS_CTL(3);
            TRACE(3, 0);
            // ---- step 3: lowest accepting label: CTA, then grid
            // (every worker warp has put its lowest accepting label into one shared-memory minimum)
            const u32 key = *(volatile u32*)&s_key;
            const u32 gmin = key == CG_NONE ? CG_NONE : key >> 5;
            const u64 gpay = key == CG_NONE ? 0ull : s_wpay[key & 31u];     // (0: the slot's fields must not overflow)
            __syncwarp();
            if (lane == 0) *(volatile u32*)&s_key = CG_NONE;          // for the next iteration (ordered by [B])
            // In scan order (CTA order starting at the CTA that holds attempt a0) every CTA holds lower
            // labels than the next one, except that CACHED the first CTA also holds the end of the window
            // in its threads below a0's ("tail" labels).  The winner is the first non-tail accept in scan
            // order; the scan stops there: slots of later CTAs are never waited for (their proposals
            // cannot win), and the first CTA, when it accepts, waits for nobody.
            const bool own_low = gmin != CG_NONE && (!CACHED || kb != 0 || gmin < tail0);
            TS_CTL(4);
            // A CTA can be up to DEPTH + 1 exchanges ahead of the slowest reader of its slot (bounded by the
            // publication check and by every fully rejected window, which needs all slots): ring of CG_SRING.
            if (nb > 1 && lane == 0)
                slot_store(my_slot + ring, ((u64)e32 << 32) | gmin,
                           ((u64)(e32 & 0xFFFFu) << 48) | ((gpay >> 32) << 24) | (gpay & 0xFFFFFFu));
            u32 q = gmin; u64 wp = gpay;
            TS_CTL(5);
            TRACE(10, 0);
            if (eq != CG_NONE) { q = eq; wp = ewp; }                   // answered before the barrier
            else if (!(own_low && kb == 0) && nb > 1) {
#ifdef CG_TRACE
                if (lane == 0) s_seg[CLS_ + 9] += 1;      // scans
#endif
                u32 tlab = CG_NONE; u64 tpay = 0;                      // tail accept of position 0
                const u32 k_end = own_low ? kb : nb;    // an accept of my own: only earlier CTAs can beat it
                u32 k0 = 0;                             // 32 scan positions at a time (measured best)
                bool found = false;
                while (!found && k0 < k_end) {
                    const u32 k = k0 + lane;
                    const bool mine = k < k_end && k != kb;
                    u32 c = c_first + k; if (c >= nb) c -= nb;
                    const u64* sl = p.slots + (size_t)(mine ? c : b) * CG_SLOT_U64 + ring;
                    bool ready = !mine; u32 l = CG_NONE; u64 q1 = 0;
                    for (;;) {
                        if (!ready) {
                            u64 q0;
                            slot_load(sl, q0, q1);
                            if ((u32)(q0 >> 32) == e32 && (u32)(q1 >> 48) == e16) {
                                ready = true; l = (u32)q0;
                                if (CACHED && k == 0 && l != CG_NONE && l >= tail0) { tlab = l; tpay = q1; l = CG_NONE; }
                            }
                        }
                        const u32 racc = __ballot_sync(CG_FULL, ready && l != CG_NONE);
                        const u32 rnot = __ballot_sync(CG_FULL, !ready);
                        const int fa = racc ? __ffs(racc) - 1 : 32;
                        const int fn = rnot ? __ffs(rnot) - 1 : 32;
                        if (fa < fn) {                  // first accepting slot, everything before it rejected
                            q = __shfl_sync(CG_FULL, l, fa);
                            wp = __shfl_sync(CG_FULL, q1, fa);
                            wp = ((wp >> 24) & 0xFFFFFFull) << 32 | (wp & 0xFFFFFFull);
                            found = true;
                            break;
                        }
                        if (!rnot) break;               // whole chunk rejected: next chunk
                    }
                    if (k0 == 0) {                      // position 0 sits in lane 0 of the first chunk
                        tlab = __shfl_sync(CG_FULL, tlab, 0); tpay = __shfl_sync(CG_FULL, tpay, 0);
                    }
                    k0 += 32;
                }
                if (!found && !own_low && kb != 0 && tlab != CG_NONE) {   // only the tail of the window accepted
                    q = tlab; wp = ((tpay >> 24) & 0xFFFFFFull) << 32 | (tpay & 0xFFFFFFull);
                }
            }
#ifdef CG_TRACE
            if (lane == 0 && !(own_low && kb == 0) && nb > 1) {       // histogram of the scan time
                const long long dt = clock64() - t_prev;
                const int bin = dt < 500 ? 11 : dt < 1000 ? 12 : dt < 2000 ? 13 : dt < 4000 ? 14 : dt < 8000 ? 1 : 2;
                s_seg[CLS_ + bin] += 1;
            }
#endif
            TRACE(4, 0);
            TS_CTL(6);
            // ---- what the workers need: attempts consumed (m = (p-1)M + q per executed hop, PAPER.md:39,
            // 78), the hop (step 3a), occupations, pending list
            const u32 used = q == CG_NONE ? M : q + 1;
            const u32 hi_ = (u32)(wp >> 32), hj_ = (u32)wp;
            const u32 ci = site_code(hi_, L), cj = site_code(hj_, L);
            if (lane == 0) *reinterpret_cast<uint4*>(&s_desc) = make_uint4(used, q != CG_NONE, ci, cj);
            // Readers start from a buffer that is complete on every CTA (hop v; this CTA's own slab of hop hl is
            // finished in the gap that ends at [B]) and add the hops v+1 .. themselves, in hop order.
            {
                const u32 hn_ = (u32)hl + (q != CG_NONE ? 1u : 0u);                 // hops executed so far
#ifdef CG_VNEW
                const u32 v = nb > 1 ? (u32)(ver - pub_base) : (u32)hl;
#else
                // one CTA: its own slab is always complete.  Several: DEPTH hops back is what the publication
                // check guarantees; starting from the newest buffer seen complete (ver) saves pending terms but
                // measured slower at 19 CTAs (-5 %) and equal at 148.
                const u32 v = nb > 1 ? (hn_ > CG_DEPTH ? hn_ - CG_DEPTH : 0u) : (u32)hl;
#endif
                const u32 np_ = hn_ - v;                                            // <= DEPTH
                if (lane == 0) {              // the workers are between the two barriers: nobody reads these
                    if (q != CG_NONE) {
                        atomicAnd(&s_n[hi_ >> 5], ~(1u << (hi_ & 31)));     // no return value: fire and forget
                        atomicOr(&s_n[hj_ >> 5], 1u << (hj_ & 31));
                        *reinterpret_cast<uint2*>(&s_pend.c[(u32)hl % CG_DEPTH][0]) = make_uint2(ci, cj);
                    }
                    *reinterpret_cast<uint4*>(&s_pend) = make_uint4(np_, (cur0 + v) % CG_RING, v % CG_DEPTH, 0u);
                }
            }
            TRACE(5, 0);
            TS_CTL(7);
            barB_arrive(TB);              // [B] the workers may read the descriptor; this warp goes on
            TS_CTL(8);
#ifdef CG_TRACE_T
            if (lane == 0 && p.trace && b < 32u && it_local - 2000u < 64u) {
                p.trace[((it_local - 2000u) * 32u + b) * 32u + 10] = kb; p.trace[((it_local - 2000u) * 32u + b) * 32u + 11] = used;
            }
#endif
            // ---- the rest of the bookkeeping, while the workers run
            if (CACHED) {
                if (t0r + used < per) t0r += used;
                else {
                    u32 g0 = c_first * per + t0r + used; if (g0 >= P) g0 -= P;      // used <= M <= P
                    c_first = g0 / per; t0r = g0 - c_first * per;
                }
                // a hint only (time to decode ahead): the workers may still see the previous value
                if (lane == 0) s_desc.ahead = c_first != b;
            }
            used_sum += used;
            ++it_local;
            if (q != CG_NONE) {
                const int xi = hi_ & (L - 1), xj = hj_ & (L - 1);
                int ddx = (xj - xi) & (L - 1); if (ddx > L / 2) ddx -= L;   // minimum image, tie -> +L/2
                dP += ddx;                                                   // step 3b: dP = dx
                if (lane == 0 && b == 0 && hops_start + hl - log_base < p.log_cap) {
                    const u64 h = hops_start + hl - log_base;
                    p.log_a[h] = a_start + used_sum - 1; p.log_i[h] = hi_; p.log_j[h] = hj_;
                }
                ++hl;
                // all slabs of hop hl - DEPTH + 1: the oldest buffer a reader may start from once the NEXT
                // hop is executed, awaited before that
                need_pub = hl >= CG_DEPTH ? pub_base + hl - CG_DEPTH + 1 : 0;
            }
            TS_CTL(9);
            TRACE(0, 0);
        }
#ifdef CG_TRACE
        __syncwarp();
        if (p.trace) { p.trace[(size_t)b * 64 + lane] += s_seg[lane]; p.trace[(size_t)b * 64 + 32 + lane] += s_seg[32 + lane]; }
#endif
#ifdef CG_TRACE_W
        if (p.trace && lane == 0) for (int k = 0; k < 16; ++k) p.trace[32768 + (size_t)b * 16 + k] = cw[k];
#endif
        if (b == 0 && lane == 0) {
            CgCtl* c = p.ctl;
            c->attempts = a_start + used_sum; c->hops = hops_start + hl;
            c->iterations += it_local; c->proposals += (u64)M * it_local;
            c->dP += dP; c->cur = (u32)((cur0 + hl) % CG_RING); c->epoch += it_local;
            c->pub_base = pub_base + hl;
            c->cyc_total += (u64)(clock64() - t_begin);
        }
        return;
    }

    Slab<TW, RP> slab;
    slab.load(p.eps[wbuf], pr0, pr1, L, (u32)tid);

    // finish the issued slab update and hand it to the service warp for publication
    auto finish_update = [&]() {
        const u32 src = wbuf == 0 ? CG_RING - 1u : wbuf - 1u;
        slab.finish(tf, mask, L, p.eps[src], p.eps[wbuf], pr0, pr1);
        if (nb > 1) barN_arrive((u32)((hl - 1) % CG_DEPTH), TB);   // hop hl (1-based) on barrier 1 + (hl - 1) % DEPTH
        upd = false;
    };

    // ---------------------------------------------------------------------- worker warps ----
    // One loop body = outcome of the previous exchange (descriptor) -> table gathers of its hop ->
    // proposals -> slab update: gathers and update sit in the same body, so the gathers stay in flight
    // during the whole propose phase.
#ifdef CG_TRACE_W
    u64 tw[7] = {}; long long wprev = 0;
#endif
    u64 a0 = a_start;                     // first attempt of the window (used when labels are not cached)
    uint4 d4 = make_uint4(0u, 0u, 0u, 0u);       // used, hop, ci, cj of the previous exchange
#ifdef CG_TRACE_T
    u32 itw = 0;
#endif
    for (;;) {
        TS_WRK(7);
        newhop = d4.y != 0;
        // the term of the hop executed last iteration for the pair I follow: the four gathers start before the
        // label bookkeeping (discarded if my attempt was consumed or theta_ij turns out to have changed)
        double a_i = 0, b_i = 0, a_j = 0, b_j = 0;
        if (CACHED && tracked && newhop) {
            a_i = __ldg(tf + ((sci - d4.w) & mask)); b_i = __ldg(tf + ((sci - d4.z) & mask));
            a_j = __ldg(tf + ((scj - d4.w) & mask)); b_j = __ldg(tf + ((scj - d4.z) & mask));
        }
        if (CACHED) {
            if (has_label && d4.x) {
                if (lab >= d4.x) lab -= d4.x;
                else {                              // my attempt was consumed: the next one, P attempts later
                    lab += P - d4.x; a_cur += P;
                    // (deferring this decode to the gap between the barriers, for attempts that re-enter far
                    // outside the window, measured slower: here it hides behind the warps that start to follow
                    // new pairs)
                    if (!nxt_valid) nxt = decode_attempt(tb, p, a_cur);
                    take(nxt); nxt_valid = false;
                }
            }
        } else a0 += d4.x;
        if (newhop) {
            // step 3b: local energies of my slab, into the next buffer of the ring
            ++hl;
            hci = d4.z; hcj = d4.w;
            wbuf = wbuf == CG_RING - 1 ? 0u : wbuf + 1u;
            upd = true;
        }
        if (hl >= p.n_hops) break;
        TS_WRK(0);
#ifdef CG_TRACE_W
        const long long w0 = clock64();
#endif
        // ---- steps 1-2: propose and test, state untouched
        u32 best = CG_NONE, bi = 0, bj = 0;
        if (CACHED) {
            const bool th = lab < M && BIT(s_n, ci_) && !BIT(s_n, cj_);   // theta_ij, inside the window
            if (th) {
                if (!tracked) {            // start to follow (i, j): complete buffer + all pending hops
                    const u32 np = s_pend.npend;
                    const double* __restrict__ erd = p.eps[s_pend.rbuf];
                    ei = ld_cg(erd + ci_); ej = ld_cg(erd + cj_);
                    for (u32 k = 0; k < np; ++k) {
                        const u32 e_ = (s_pend.first + k) % CG_DEPTH;
                        const u32 ki = s_pend.c[e_][0], kj = s_pend.c[e_][1];
                        ei = __dadd_rn(ei, hop_term(tf, mask, sci, ki, kj));
                        ej = __dadd_rn(ej, hop_term(tf, mask, scj, ki, kj));
                    }
                    tracked = true;
                } else if (newhop) {       // the term of the hop executed last iteration (gathered above)
                    ei = __dadd_rn(ei, __dsub_rn(a_i, b_i)); ej = __dadd_rn(ej, __dsub_rn(a_j, b_j));
                }
                // dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
                const double dE = __dsub_rn(__dsub_rn(__dsub_rn(ej, ei), c_invr), c_fld);
                if (metropolis(dE, cuh, cul, p.T, p.inv_T)) { best = lab; bi = ci_; bj = cj_; }
            } else tracked = false;
        } else {
            const u32 np = s_pend.npend;
            const double* __restrict__ erd = p.eps[s_pend.rbuf];
            for (u32 l = lab0 + tid; l < lab1; l += TW) {
                const u64 a = a0 + l;
                u32 w0, w1, w2, w3;
                philox4x32_10((u32)a, (u32)(a >> 32), 0u, 0u, p.seed_lo, p.seed_hi, w0, w1, w2, w3);
                const u32 i = __umulhi(w0, N);                                   // uniform site
                if (!BIT(s_n, i)) continue;                                      // n_i = 1 ?
                const u32 k = tower_search(tb, ((u64)w1 << 11) | (u64)(w2 >> 21));
                const u32 j = hop_target(tb, i, k, L, lg);
                if (BIT(s_n, j)) continue;                                       // n_j = 0 ?
                double vi = ld_cg(erd + i), vj = ld_cg(erd + j);
                const u32 si = site_code(i, L) | (u32)L, sj = site_code(j, L) | (u32)L;
                for (u32 t = 0; t < np; ++t) {
                    const u32 e_ = (s_pend.first + t) % CG_DEPTH;
                    const u32 ki = s_pend.c[e_][0], kj = s_pend.c[e_][1];
                    vi = __dadd_rn(vi, hop_term(tf, mask, si, ki, kj));
                    vj = __dadd_rn(vj, hop_term(tf, mask, sj, ki, kj));
                }
                const double dE = __dsub_rn(__dsub_rn(__dsub_rn(vj, vi), s_invr[k]), s_fld[k]);
                if (metropolis(dE, w2 & 0x1FFFFFu, w3, p.T, p.inv_T)) { best = l; bi = i; bj = j; break; }
            }
        }
        TS_WRK(1);
#ifdef CG_TRACE_W
        const long long w1 = clock64();
#endif
        // ---- step 3: lowest accepting label: warp, then the control warp
        {
            const u32 wmin = __reduce_min_sync(CG_FULL, best);
            if (wmin != CG_NONE && best == wmin) {     // labels are distinct: one lane
                s_wpay[warp] = ((u64)bi << 32) | (u64)bj;
                atomicMin(&s_key, (wmin << 5) | (u32)warp);
            }
        }
        TS_WRK(2);
#ifdef CG_TRACE_W
        const long long w2 = clock64();
#endif
        barX_arrive(TB);                  // [A] only the control warp waits here: the workers go on to their slabs
        TS_WRK(3);
#ifdef CG_TRACE_W
        const long long w3 = clock64();
#endif
        // while the control warp does the exchange: the slab of the previous hop (its table gathers,
        // issued when that hop was executed, have had the whole propose phase to arrive) and, if another
        // CTA holds the start of the window, the decode one attempt ahead
        if (upd) slab.issue(tf, mask, pr0, pr1, hci, hcj);
        if (has_label && !nxt_valid) { nxt = decode_attempt(tb, p, a_cur + P); nxt_valid = true; }   // behind the gathers
        if (upd) finish_update();
        TS_WRK(4);
#ifdef CG_TRACE_W
        const long long w4 = clock64();
#endif
        barB_sync(TB);                    // [B] the control warp has written the descriptor
        TS_WRK(5);
#ifdef CG_TRACE_W
        {
            const long long w5 = clock64();
            tw[0] += (u64)(w1 - w0); tw[1] += (u64)(w2 - w1); tw[2] += (u64)(w3 - w2); tw[3] += (u64)(w4 - w3); tw[4] += (u64)(w5 - w4);
            if (wprev) tw[5] += (u64)(w0 - wprev);
            wprev = w5; ++tw[6];
        }
#endif
        d4 = *reinterpret_cast<const uint4*>(&s_desc);      // used, hop, ci, cj
        ahead = s_desc.ahead != 0;
        TS_WRK(6);
#ifdef CG_TRACE_T
        ++itw;
#endif
    }
#ifdef CG_TRACE_W
    if (p.trace && lane == 0) for (int k = 0; k < 7; ++k) p.trace[((size_t)b * 16 + warp) * 8 + k] = tw[k];
#endif
    if (upd) { slab.issue(tf, mask, pr0, pr1, hci, hcj); finish_update(); }
    if (b == 0)
        for (u32 w = tid; w < (N + 31) / 32; w += TW) p.nbits[w] = s_n[w];
}

template <int THREADS, int RP, bool CACHED>
__global__ void __launch_bounds__(THREADS, 1) cg_pr_persistent(const CgParams p)
{
    pr_persistent_body<THREADS, RP, CACHED>(p, blockIdx.x, gridDim.x);
}

// Replica packing (the paper recommends averaging many samples): ONE launch,
// CTAs [first[s], first[s+1]) run sim s with its own parameter block.  The sims share nothing.
template <int THREADS, int RP, bool CACHED>
__global__ void __launch_bounds__(THREADS, 1)
cg_pr_persistent_many(const CgParams* __restrict__ ps, const u32* __restrict__ first, const u32 n_sims)
{
    __shared__ CgParams sp;
    __shared__ u32 s_b, s_nb;
    if (threadIdx.x == 0) {
        u32 s = 0;
        while (s + 1 < n_sims && first[s + 1] <= blockIdx.x) ++s;
        s_b = blockIdx.x - first[s]; s_nb = first[s + 1] - first[s];
        sp = ps[s];
    }
    __syncthreads();
    pr_persistent_body<THREADS, RP, CACHED>(sp, s_b, s_nb);
}

// Step a6 alone: scripted hops, update in place (no readers), one launch.
template <int THREADS, int RP>
__global__ void __launch_bounds__(THREADS, 1)
cg_update_scripted(const CgParams p, const u32* __restrict__ hop_i, const u32* __restrict__ hop_j, u64 count)
{
    const u32 b = blockIdx.x, nb = gridDim.x;
    const int L = p.L;
    const u32 mask = ((u32)(L - 1) << (p.lgL + 1)) | (u32)(L - 1);
    const u32 pairs = p.N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    double* e = p.eps[p.ctl->cur];
    Slab<THREADS, RP> slab;
    slab.load(e, pr0, pr1, L, threadIdx.x);
    for (u64 h = 0; h < count; ++h) {
        slab.issue(p.tf, mask, pr0, pr1, site_code(__ldg(hop_i + h), L), site_code(__ldg(hop_j + h), L));
        slab.finish(p.tf, mask, L, e, e, pr0, pr1);
    }
    if (b == 0 && threadIdx.x == 0) {       // occupations and dipole moment, in hop order
        long long dP = p.ctl->dP; u32 bad = 0;
        for (u64 h = 0; h < count; ++h) {
            const u32 i = hop_i[h], j = hop_j[h];
            const u32 wi = p.nbits[i >> 5], wj = p.nbits[j >> 5];
            if (!((wi >> (i & 31)) & 1u) || ((wj >> (j & 31)) & 1u)) ++bad;
            p.nbits[i >> 5] &= ~(1u << (i & 31));
            p.nbits[j >> 5] |= (1u << (j & 31));
            int ddx = ((int)(j & (L - 1)) - (int)(i & (L - 1))) & (L - 1); if (ddx > L / 2) ddx -= L;
            dP += ddx;
        }
        p.ctl->dP = dP; p.ctl->hops += count; p.ctl->bad_hops += bad;
    }
}

// tf from the quarter table (one-time set-up)
__global__ void cg_build_tf(const double* __restrict__ tq, double* __restrict__ tf, int L, int pitch)
{
    const int dy = blockIdx.x;
    const int fy = min(dy, L - dy);
    for (int dx = threadIdx.x; dx <= L; dx += blockDim.x) {
        const int w = dx & (L - 1), fx = min(w, L - w);
        tf[(size_t)dy * 2 * L + dx] = tq[fy * pitch + fx];
    }
}

// ---- one-time set-up (step a0) --------------------------------------------------------------

// phi_s = (u - 1/2) W with u from Philox domain 1; occupation key from domain 2.
__global__ void cg_init_phi_keys(double* phi, u64* keys, u32 N, double W, u32 seed_lo, u32 seed_hi)
{
    const u32 s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    u32 w0, w1, w2, w3;
    philox4x32_10(s, 0u, 1u, 0u, seed_lo, seed_hi, w0, w1, w2, w3);
    const double u = (double)((((u64)w0 << 32) | (u64)w1) >> 11) * (1.0 / 9007199254740992.0);
    phi[s] = __dmul_rn(__dsub_rn(u, 0.5), W);
    philox4x32_10(s, 0u, 2u, 0u, seed_lo, seed_hi, w0, w1, w2, w3);
    keys[s] = ((u64)w0 << 32) | (u64)w1;
}

// n_s = 1 for the N/2 sites with the smallest (key, s): rank by counting.
__global__ void cg_init_occupations(const u64* __restrict__ keys, u32* nbits, u32 N)
{
    __shared__ u64 tile[1024];
    const u32 s = blockIdx.x * blockDim.x + threadIdx.x;       // N is a multiple of blockDim
    const u64 mine = keys[s];
    u32 rank = 0;
    for (u32 t0 = 0; t0 < N; t0 += blockDim.x) {
        tile[threadIdx.x] = keys[t0 + threadIdx.x];
        __syncthreads();
        for (u32 k = 0; k < blockDim.x; ++k) {
            const u64 other = tile[k];
            rank += (other < mine) || (other == mine && t0 + k < s);
        }
        __syncthreads();
    }
    const u32 word = __ballot_sync(__activemask(), rank < N / 2);
    if ((threadIdx.x & 31) == 0) nbits[s >> 5] = word;
}

// eps_s = phi_s + sum_{t != s} (n_t - 1/2)/r_st in index order t.
__global__ void cg_full_sum_eps(const double* __restrict__ phi, const u32* __restrict__ nbits,
                                const double* __restrict__ tq, double* __restrict__ out,
                                int L, int lg, int pitch, u32 N)
{
    const u32 s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int y = s >> lg, x = s & (L - 1);
    double e = phi[s];
    u32 word = 0;
    for (int yt = 0; yt < L; ++yt) {
        int dy = (y - yt) & (L - 1); dy = min(dy, L - dy);
        const double* row = tq + dy * pitch;
        for (int xt = 0; xt < L; ++xt) {
            const u32 t = ((u32)yt << lg) | (u32)xt;
            if ((t & 31u) == 0u || xt == 0) word = __ldg(nbits + (t >> 5));
            int dx = (x - xt) & (L - 1); dx = min(dx, L - dx);
            const double half = __dmul_rn(0.5, __ldg(row + dx));  // exact; 0 on the diagonal
            e = ((word >> (t & 31u)) & 1u) ? __dadd_rn(e, half) : __dsub_rn(e, half);
        }
    }
    out[s] = e;
}

__global__ void cg_max_abs_diff(const double* a, const double* b, u32 N, u64* out_bits)
{
    double m = 0.0;
    for (u32 s = blockIdx.x * blockDim.x + threadIdx.x; s < N; s += gridDim.x * blockDim.x)
        m = fmax(m, fabs(a[s] - b[s]));
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(CG_FULL, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out_bits, (u64)__double_as_longlong(m)); // m >= 0
}

// L2 roofline probe: L1-bypassing 16-byte read-modify-write over a resident buffer.
__global__ void __launch_bounds__(512) cg_l2_rmw(double2* buf, size_t n16, int reps)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r)
        for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n16; k += stride) {
            double2 v = __ldcg(buf + k);
            v.x += 1.0; v.y -= 1.0;
            __stcg(buf + k, v);
        }
}

// -------------------------------------------------------------------- host --

struct cg_sim {
    int L = 0, lgL = 0, pitch = 0;
    u32 N = 0, M = 0;
    double W = 0, xi = 0, T = 0, E = 0;
    u64 seed = 0;
    // host tables (live part of the tower)
    int64_t K = 0, Klive = 0;
    std::vector<int32_t> dy, dx;
    std::vector<double> cdf, invr_k, fld_k;
    std::vector<u64> cdfi;
    std::vector<u32> guide;
    double S = 0, Gamma = 0;
    // device
    cudaStream_t stream = nullptr;
    void* ws = nullptr; bool own_ws = false;
    double* d_eps[CG_RING] = {};
    double* d_scratch = nullptr; double* d_phi = nullptr;
    u32* d_nbits = nullptr; double* d_tq = nullptr; double* d_tf = nullptr;
    u64* d_cdfi = nullptr; double* d_invr_k = nullptr; double* d_fld_k = nullptr; int* d_disp = nullptr;
    u32* d_guide = nullptr;
    u64* d_slots = nullptr; CgCtl* d_ctl = nullptr; u64* d_red = nullptr;
    void* d_log = nullptr; bool own_log = false; u64 log_cap = 0;
    bool log_gap = false;                 // scripted hops (cg_apply_hops) were executed while the log was on: it no longer holds every hop
    u64* d_trace = nullptr; u32 trace_iters = 0;
    void* d_many = nullptr; size_t many_cap = 0;      // parameter blocks of cg_run_many (owned by its first sim)
    // launch shape
    int num_sms = 0, n_ctas = 0, threads = 0, smem = 0, rp = 0, pl = 0;   // pl > 0: cached proposals
    std::string err;
};

static int fail_cuda(cg_sim* s, cudaError_t e, const char* what)
{
    if (s) {
        char buf[256];
        snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
        s->err = buf;
    }
    return CG_ECUDA;
}
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail_cuda(s, e__, #call); } while (0)
#define CK0(sim, call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail_cuda(sim, e__, #call); } while (0)

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool valid_L(int L, int* lg)
{
    if (L < 4 || L > 1024 || (L & (L - 1))) return false;
    int k = 0; while ((1 << k) < L) ++k;
    if (lg) *lg = k;
    return true;
}

struct WsLayout { size_t eps0, scratch, phi, nbits, tq, tf, cdfi, invr_k, fld_k, disp, guide, slots, ctl, red, total; };
#define CG_SLOT_BYTES ((size_t)8 * CG_SLOT_U64 * CG_MAX_CTAS)

static WsLayout ws_layout(int L)
{
    const size_t N = (size_t)L * L, h = (size_t)L / 2 + 1;
    WsLayout w; size_t o = 0;
    w.eps0 = o; o += CG_RING * align256(8 * N);
    w.scratch = o; o += align256(8 * N);
    w.phi = o; o += align256(8 * N);
    w.nbits = o; o += align256(N / 8 + 4);
    w.tq = o; o += align256(8 * h * h);
    w.tf = o; o += align256(16 * N);
    w.cdfi = o; o += align256(8 * N);           // tower can never be longer than N entries
    w.invr_k = o; o += align256(8 * N);
    w.fld_k = o; o += align256(8 * N);
    w.disp = o; o += align256(4 * N);
    w.guide = o; o += align256(4 * CG_GUIDE);
    w.slots = o; o += align256(CG_SLOT_BYTES);
    w.ctl = o; o += align256(sizeof(CgCtl));
    w.red = o; o += 256;
    w.total = o;
    return w;
}

extern "C" size_t cg_workspace_bytes(int L, uint32_t M)
{
    (void)M;
    if (!valid_L(L, nullptr)) return 0;
    return ws_layout(L).total;
}

// Displacement list, tower and Gamma on the host.
static void build_tables(cg_sim* s, std::vector<double>& tq)
{
    const int L = s->L, h = L / 2;
    struct D { long long r2; int dy, dx; };
    std::vector<D> d;
    for (int dy = -h + 1; dy <= h; ++dy)
        for (int dx = -h + 1; dx <= h; ++dx) {
            const long long r2 = (long long)dy * dy + (long long)dx * dx;
            if (r2 > 0 && r2 <= (long long)h * h) d.push_back({r2, dy, dx});
        }
    std::sort(d.begin(), d.end(), [](const D& a, const D& b) {
        if (a.r2 != b.r2) return a.r2 < b.r2;
        if (a.dy != b.dy) return a.dy < b.dy;
        return a.dx < b.dx;
    });
    const size_t K = d.size();
    std::vector<double> run(K);
    double acc = 0.0;
    for (size_t k = 0; k < K; ++k) {
        const double r = std::sqrt((double)d[k].r2);
        const double t = -2.0 * r;
        acc = acc + std::exp(t / s->xi);
        run[k] = acc;
    }
    s->K = (int64_t)K; s->S = acc; s->Gamma = (double)s->N * acc;
    size_t live = K;
    for (size_t k = 0; k < K; ++k) {
        const double c = (k + 1 == K) ? 1.0 : run[k] / acc;
        if (c >= 1.0) { live = k + 1; break; }
    }
    s->Klive = (int64_t)live;
    s->dy.resize(live); s->dx.resize(live); s->cdf.resize(live); s->invr_k.resize(live);
    s->fld_k.resize(live); s->cdfi.resize(live);
    for (size_t k = 0; k < live; ++k) {
        s->dy[k] = d[k].dy; s->dx[k] = d[k].dx;
        s->cdf[k] = (k + 1 == K) ? 1.0 : run[k] / acc;
        s->invr_k[k] = 1.0 / std::sqrt((double)d[k].r2);
        s->fld_k[k] = s->E * (double)d[k].dx;              // the field term of dH
    }
    s->cdf[live - 1] = 1.0;
    // u_d = m 2^-43 with integer m < 2^43, so u_d < cdf_k <=> m < ceil(cdf_k 2^43) (scaling by a power
    // of two and ceil are exact in double)
    for (size_t k = 0; k < live; ++k) s->cdfi[k] = (u64)std::ceil(std::ldexp(s->cdf[k], 43));
    // Guide over t = 2^43 - m: bucket = (binade of t, next 3 bits).  The tail of the tower is geometric
    // in r, so every bucket brackets only a few k; both ends found by the plain search.
    auto kstar = [&](u64 m) { size_t k = 0; while (!(m < s->cdfi[k])) ++k; return (u32)k; };
    s->guide.assign(CG_GUIDE, 0u);
    for (int e = 0; e <= 43; ++e)
        for (int mant = 0; mant < 8; ++mant) {
            u64 tlo, thi;
            if (e >= 3) { tlo = (u64)(8 + mant) << (e - 3); thi = (((u64)(8 + mant + 1)) << (e - 3)) - 1; }
            else { if (mant & ((1 << (3 - e)) - 1)) continue; tlo = thi = (u64)(8 + mant) >> (3 - e); }
            const u64 top = 1ull << 43;
            if (tlo > top) continue;
            if (thi > top) thi = top;
            const u32 klo = kstar(top - thi), khi = kstar(top - tlo);
            s->guide[(size_t)e * 8 + mant] = klo | (khi << 16);
        }
    const int pitch = s->pitch;
    tq.assign((size_t)pitch * pitch, 0.0);
    for (int a = 0; a <= h; ++a)
        for (int b = 0; b <= h; ++b) {
            const long long r2 = (long long)a * a + (long long)b * b;
            tq[(size_t)a * pitch + b] = r2 ? 1.0 / std::sqrt((double)r2) : 0.0;
        }
}

static size_t smem_bytes(const cg_sim* s)
{
    return (size_t)s->Klive * 28 + 4 * CG_GUIDE + 4 * (((size_t)s->N + 31) / 32) + 16;
}

static CgParams make_params(const cg_sim* s, u64 n_hops)
{
    CgParams p;
    for (int k = 0; k < CG_RING; ++k) p.eps[k] = s->d_eps[k];
    p.tf = s->d_tf; p.tq = s->d_tq; p.nbits = s->d_nbits;
    p.cdfi = s->d_cdfi; p.invr_k = s->d_invr_k; p.fld_k = s->d_fld_k; p.disp = s->d_disp;
    p.guide = s->d_guide;
    p.slots = s->d_slots; p.ctl = s->d_ctl;
    p.log_a = (u64*)s->d_log;
    p.log_i = s->d_log ? (u32*)((char*)s->d_log + 8 * s->log_cap) : nullptr;
    p.log_j = s->d_log ? (u32*)((char*)s->d_log + 12 * s->log_cap) : nullptr;
    p.log_cap = s->d_log ? s->log_cap : 0;
    p.L = s->L; p.lgL = s->lgL; p.pitch = s->pitch; p.Klive = (int)s->Klive;
    p.N = s->N; p.M = s->M; p.PL = (u32)s->pl;
    p.seed_lo = (u32)s->seed; p.seed_hi = (u32)(s->seed >> 32);
    p.T = s->T; p.E = s->E; p.inv_T = (float)(1.0 / s->T); p.n_hops = n_hops;
    p.trace = s->d_trace; p.trace_iters = s->trace_iters;
    return p;
}

typedef void (*persist_fn)(const CgParams);
typedef void (*scripted_fn)(const CgParams, const u32*, const u32*, u64);

// RP = eps pairs a thread keeps in registers (0: the slab streams through global memory)
template <int THREADS, bool CACHED>
static persist_fn persistent_kernel_t(int rp)
{
    switch (rp) {
        case 0: return cg_pr_persistent<THREADS, 0, CACHED>;
        case 1: return cg_pr_persistent<THREADS, 1, CACHED>;
        case 2: return cg_pr_persistent<THREADS, 2, CACHED>;
        case 4: return cg_pr_persistent<THREADS, 4, CACHED>;
        case 8: return cg_pr_persistent<THREADS, 8, CACHED>;
    }
    return nullptr;
}
static persist_fn persistent_kernel(int threads, int rp, bool cached)
{
    switch (threads) {
        case 256: return cached ? persistent_kernel_t<256, true>(rp) : persistent_kernel_t<256, false>(rp);
        case 512: return cached ? persistent_kernel_t<512, true>(rp) : persistent_kernel_t<512, false>(rp);
        case 1024: if (rp > 2) return nullptr;
                   return cached ? persistent_kernel_t<1024, true>(rp) : persistent_kernel_t<1024, false>(rp);
    }
    return nullptr;
}
typedef void (*many_fn)(const CgParams*, const u32*, u32);
template <bool CACHED>
static many_fn many_kernel_t(int rp)
{
    switch (rp) {
        case 0: return cg_pr_persistent_many<512, 0, CACHED>;
        case 1: return cg_pr_persistent_many<512, 1, CACHED>;
        case 2: return cg_pr_persistent_many<512, 2, CACHED>;
        case 4: return cg_pr_persistent_many<512, 4, CACHED>;
        case 8: return cg_pr_persistent_many<512, 8, CACHED>;
    }
    return nullptr;
}
static many_fn many_kernel(int threads, int rp, bool cached)
{
    if (threads != 512) return nullptr;
    return cached ? many_kernel_t<true>(rp) : many_kernel_t<false>(rp);
}
static scripted_fn scripted_kernel(int rp)
{
    switch (rp) {
        case 0: return cg_update_scripted<512, 0>;
        case 1: return cg_update_scripted<512, 1>;
        case 2: return cg_update_scripted<512, 2>;
        case 4: return cg_update_scripted<512, 4>;
        case 8: return cg_update_scripted<512, 8>;
    }
    return nullptr;
}

// smallest supported register tiling that holds `pairs` pairs per CTA, else 0 (streaming)
static int choose_rp(u64 pairs, int n_ctas, int threads)
{
    const u64 per_cta = (pairs + n_ctas - 1) / n_ctas;
    const u64 workers = (u64)threads - 64;               // the last two warps of a CTA hold no eps
    const u64 need = (per_cta + workers - 1) / workers;
    const int cap = threads == 1024 ? 2 : 8;
    for (int rp = 1; rp <= cap; rp *= 2)
        if ((u64)rp >= need) return rp;
    return 0;
}

static int max_coresident(cg_sim* s, int threads, int rp, bool cached, int* out)
{
    persist_fn f = persistent_kernel(threads, rp, cached);
    if (!f) return CG_EINVAL;
    CK(cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem));
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)f, threads, s->smem));
    *out = std::min(per_sm * s->num_sms, CG_MAX_CTAS);
    return CG_OK;
}

// threads per CTA that own attempts when the proposals can be cached (M <= n_ctas * pl), else 0
static int choose_pl(u64 M, int n_ctas, int threads)
{
    return M <= (u64)n_ctas * (u64)(threads - 64) ? threads - 64 : 0;
}

static int choose_launch(cg_sim* s, int n_ctas, int threads)
{
    if (threads == 0) threads = 512;
    if (threads != 256 && threads != 512 && threads != 1024) return CG_EINVAL;
    const bool heuristic = n_ctas == 0;
    if (heuristic) {
        const u64 work = std::max<u64>(s->M, s->N / 2);        // labels or pairs of sites, per worker thread
        const u64 workers = (u64)threads - 64;
        n_ctas = (int)std::min<u64>((work + workers - 1) / workers, (u64)s->num_sms);
        n_ctas = std::max(1, n_ctas);
    }
    if (n_ctas < 1 || n_ctas > CG_MAX_CTAS) return CG_EINVAL;
    int rp = choose_rp(s->N / 2, n_ctas, threads), pl = choose_pl(s->M, n_ctas, threads);
    int cap = 0;
    int rc = max_coresident(s, threads, rp, pl > 0, &cap);
    if (rc != CG_OK) return rc;
    if (cap < 1) { s->err = "persistent kernel does not fit on an SM"; return CG_EUNSUPPORTED; }
    if (n_ctas > cap) {
        if (!heuristic) return CG_EINVAL;
        n_ctas = cap;
        rp = choose_rp(s->N / 2, n_ctas, threads); pl = choose_pl(s->M, n_ctas, threads);
        rc = max_coresident(s, threads, rp, pl > 0, &cap);
        if (rc != CG_OK) return rc;
        if (n_ctas > cap) return CG_EUNSUPPORTED;
    }
    if (n_ctas != s->n_ctas)   // slots of CTAs that no longer exist must not look published
        CK(cudaMemsetAsync(s->d_slots, 0, CG_SLOT_BYTES, s->stream));
    s->n_ctas = n_ctas; s->threads = threads; s->rp = rp; s->pl = pl;
    return CG_OK;
}

static int init_impl(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed,
                     uint32_t M, void* dev_ws, size_t bytes, void* stream, bool own)
{
    if (!out) return CG_EINVAL;
    *out = nullptr;
    if (L < 2 || (L & 1)) return CG_EINVAL;
    if (!(xi > 0.0) || !(T > 0.0) || !(W >= 0.0) || M < 1 || !std::isfinite(E) || !std::isfinite(W)
        || !std::isfinite(xi) || !std::isfinite(T)) return CG_EINVAL;
    int lg = 0;
    if (!valid_L(L, &lg)) return CG_EUNSUPPORTED;
    cg_sim* s = new (std::nothrow) cg_sim();
    if (!s) return CG_ENOMEM;
    struct Guard { cg_sim* s; ~Guard() { if (s) cg_free(s); } } guard{s};
    s->L = L; s->lgL = lg; s->pitch = L / 2 + 1; s->N = (u32)L * (u32)L; s->M = M;
    s->W = W; s->xi = xi; s->T = T; s->E = E; s->seed = seed;
    s->stream = (cudaStream_t)stream;

    int dev = 0;
    cudaDeviceProp prop;
    CK(cudaGetDevice(&dev));
    CK(cudaGetDeviceProperties(&prop, dev));
    s->num_sms = prop.multiProcessorCount;
    if (!prop.cooperativeLaunch) { s->err = "device lacks cooperative launch"; return CG_EUNSUPPORTED; }

    std::vector<double> tq;
    try { build_tables(s, tq); } catch (const std::bad_alloc&) { return CG_ENOMEM; }
    if (s->Klive > 65535) return CG_EUNSUPPORTED;           // the guide packs k in 16 bits
    s->smem = (int)smem_bytes(s);
    if ((size_t)s->smem > (size_t)prop.sharedMemPerBlockOptin - 1024) return CG_EUNSUPPORTED;

    const WsLayout w = ws_layout(L);
    if (own) {
        CK(cudaMalloc(&s->ws, w.total));
        s->own_ws = true;
    } else {
        if (!dev_ws || ((uintptr_t)dev_ws & 255)) return CG_EINVAL;
        if (bytes < w.total) return CG_ENOMEM;
        s->ws = dev_ws;
    }
    char* base = (char*)s->ws;
    for (int k = 0; k < CG_RING; ++k) s->d_eps[k] = (double*)(base + w.eps0 + (size_t)k * align256(8 * (size_t)s->N));
    s->d_scratch = (double*)(base + w.scratch); s->d_phi = (double*)(base + w.phi);
    s->d_nbits = (u32*)(base + w.nbits); s->d_tq = (double*)(base + w.tq); s->d_tf = (double*)(base + w.tf);
    s->d_cdfi = (u64*)(base + w.cdfi); s->d_invr_k = (double*)(base + w.invr_k);
    s->d_fld_k = (double*)(base + w.fld_k); s->d_guide = (u32*)(base + w.guide);
    s->d_disp = (int*)(base + w.disp); s->d_slots = (u64*)(base + w.slots);
    s->d_ctl = (CgCtl*)(base + w.ctl); s->d_red = (u64*)(base + w.red);

    std::vector<int> disp((size_t)s->Klive);
    for (int64_t k = 0; k < s->Klive; ++k) disp[k] = (s->dy[k] << 16) | (s->dx[k] & 0xFFFF);
    cudaStream_t st = s->stream;
    CK(cudaMemcpyAsync(s->d_tq, tq.data(), 8 * tq.size(), cudaMemcpyHostToDevice, st));
    cg_build_tf<<<L, 256, 0, st>>>(s->d_tq, s->d_tf, L, s->pitch);
    CK(cudaMemcpyAsync(s->d_cdfi, s->cdfi.data(), 8 * (size_t)s->Klive, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(s->d_invr_k, s->invr_k.data(), 8 * (size_t)s->Klive, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(s->d_fld_k, s->fld_k.data(), 8 * (size_t)s->Klive, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(s->d_guide, s->guide.data(), 4 * (size_t)CG_GUIDE, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(s->d_disp, disp.data(), 4 * (size_t)s->Klive, cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(s->d_slots, 0, CG_SLOT_BYTES, st));
    CgCtl ctl; memset(&ctl, 0, sizeof ctl); ctl.epoch = 1;
    CK(cudaMemcpyAsync(s->d_ctl, &ctl, sizeof ctl, cudaMemcpyHostToDevice, st));

    // disorder, occupations, local energies
    const u32 N = s->N;
    const int tb = (int)std::min<u32>(N, 256);
    u64* keys = (u64*)s->d_eps[1];
    cg_init_phi_keys<<<(N + tb - 1) / tb, tb, 0, st>>>(s->d_phi, keys, N, W, (u32)seed, (u32)(seed >> 32));
    const int ob = (int)std::min<u32>(N, 1024);          // N = 4^k >= 16, so ob divides N and is a warp multiple
    cg_init_occupations<<<N / ob, ob, 0, st>>>(keys, s->d_nbits, N);
    cg_full_sum_eps<<<(N + 127) / 128, 128, 0, st>>>(s->d_phi, s->d_nbits, s->d_tq, s->d_eps[0], L, lg, s->pitch, N);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));                        // host vectors above go out of scope

    int rc = choose_launch(s, 0, 0);
    if (rc != CG_OK) return rc;
    guard.s = nullptr;
    *out = s;
    return CG_OK;
}

extern "C" int cg_init(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed, uint32_t M)
{
    return init_impl(out, L, W, xi, T, E, seed, M, nullptr, 0, nullptr, true);
}

extern "C" int cg_init_ws(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed,
                          uint32_t M, void* dev_workspace, size_t bytes, void* cuda_stream)
{
    return init_impl(out, L, W, xi, T, E, seed, M, dev_workspace, bytes, cuda_stream, false);
}

extern "C" void cg_free(cg_sim* s)
{
    if (!s) return;
    if (s->stream || s->ws) cudaStreamSynchronize(s->stream);
    if (s->own_log && s->d_log) cudaFree(s->d_log);
    if (s->d_many) cudaFree(s->d_many);
    if (s->own_ws && s->ws) cudaFree(s->ws);
    delete s;
}

extern "C" int cg_run(cg_sim* s, uint64_t n_hops)
{
    if (!s) return CG_EINVAL;
    if (n_hops == 0) return CG_OK;
    persist_fn f = persistent_kernel(s->threads, s->rp, s->pl > 0);
    if (!f) return CG_EINVAL;
    CgParams p = make_params(s, n_hops);
    void* args[] = {&p};
    CK(cudaLaunchCooperativeKernel((const void*)f, dim3(s->n_ctas), dim3(s->threads), args, (size_t)s->smem, s->stream));
    return CG_OK;
}

extern "C" int cg_run_many(cg_sim* const* sims, int n_sims, uint64_t n_hops)
{
    if (!sims || n_sims < 1 || n_sims > CG_MAX_CTAS) return CG_EINVAL;
    cg_sim* s0 = sims[0];
    if (!s0) return CG_EINVAL;
    if (n_hops == 0) return CG_OK;
    std::vector<CgParams> ps((size_t)n_sims);
    std::vector<u32> first((size_t)n_sims + 1, 0u);
    int smem = 0;
    for (int k = 0; k < n_sims; ++k) {
        cg_sim* s = sims[k];
        if (!s) return CG_EINVAL;
        for (int m = 0; m < k; ++m) if (sims[m] == s) return CG_EINVAL;       // a sim may appear once
        if (s->stream != s0->stream || s->threads != s0->threads || s->rp != s0->rp || (s->pl > 0) != (s0->pl > 0)) {
            s0->err = "cg_run_many: the sims must share stream and launch shape (threads, register tiling, cached labels)";
            return CG_EINVAL;
        }
        ps[(size_t)k] = make_params(s, n_hops);
        first[(size_t)k + 1] = first[(size_t)k] + (u32)s->n_ctas;
        smem = std::max(smem, s->smem);
    }
    many_fn f = many_kernel(s0->threads, s0->rp, s0->pl > 0);
    if (!f) { s0->err = "cg_run_many: only 512-thread launch shapes"; return CG_EUNSUPPORTED; }
    CK0(s0, cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int per_sm = 0;
    CK0(s0, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)f, s0->threads, smem));
    const u32 total = first[(size_t)n_sims];
    if (total > (u32)(per_sm * s0->num_sms)) {     // every CTA of every sim must be resident: they wait for each other
        s0->err = "cg_run_many: the sims' CTAs do not fit on the device together";
        return CG_EUNSUPPORTED;
    }
    const size_t need = ps.size() * sizeof(CgParams) + first.size() * sizeof(u32);
    if (s0->many_cap < need) {
        if (s0->d_many) { CK0(s0, cudaStreamSynchronize(s0->stream)); cudaFree(s0->d_many); s0->d_many = nullptr; s0->many_cap = 0; }
        CK0(s0, cudaMalloc(&s0->d_many, need));
        s0->many_cap = need;
    }
    CgParams* d_ps = (CgParams*)s0->d_many;
    u32* d_first = (u32*)((char*)s0->d_many + ps.size() * sizeof(CgParams));
    // pageable sources: the copies are staged before the calls return
    CK0(s0, cudaMemcpyAsync(d_ps, ps.data(), ps.size() * sizeof(CgParams), cudaMemcpyHostToDevice, s0->stream));
    CK0(s0, cudaMemcpyAsync(d_first, first.data(), first.size() * sizeof(u32), cudaMemcpyHostToDevice, s0->stream));
    u32 n = (u32)n_sims;
    void* args[] = {&d_ps, &d_first, &n};
    CK0(s0, cudaLaunchCooperativeKernel((const void*)f, dim3(total), dim3(s0->threads), args, (size_t)smem, s0->stream));
    return CG_OK;
}

static int read_ctl(cg_sim* s, CgCtl* c)
{
    CK(cudaMemcpyAsync(c, s->d_ctl, sizeof *c, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_get_state(cg_sim* s, int8_t* n, double* eps, double* t_tau0, int64_t* dP)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (eps) CK(cudaMemcpyAsync(eps, s->d_eps[c.cur % CG_RING], 8 * (size_t)s->N, cudaMemcpyDeviceToHost, s->stream));
    if (n) {
        std::vector<u32> bits((s->N + 31) / 32);
        CK(cudaMemcpyAsync(bits.data(), s->d_nbits, 4 * bits.size(), cudaMemcpyDeviceToHost, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        for (u32 k = 0; k < s->N; ++k) n[k] = (int8_t)((bits[k >> 5] >> (k & 31)) & 1u);
    }
    CK(cudaStreamSynchronize(s->stream));
    if (t_tau0) *t_tau0 = (double)c.attempts / s->Gamma;     // deterministic dt = m/Gamma
    if (dP) *dP = c.dP;
    return CG_OK;
}

extern "C" int cg_set_state(cg_sim* s, const int8_t* n, const double* eps, uint64_t attempts,
                            uint64_t hops, int64_t dP)
{
    if (!s || !n || !eps) return CG_EINVAL;
    std::vector<u32> bits((s->N + 31) / 32, 0u);
    u64 sum = 0;
    for (u32 k = 0; k < s->N; ++k) {
        if (n[k] != 0 && n[k] != 1) return CG_EINVAL;
        sum += (u64)n[k];
        bits[k >> 5] |= (u32)n[k] << (k & 31);
    }
    if (sum != s->N / 2) return CG_EINVAL;                   // sum_i n_i = nu N
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    c.attempts = attempts; c.hops = hops; c.dP = dP; c.iterations = 0; c.proposals = 0; c.cur = 0;
    c.log_base = hops; c.log_a0 = attempts; s->log_gap = false;
    CK(cudaMemcpyAsync(s->d_eps[0], eps, 8 * (size_t)s->N, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(s->d_nbits, bits.data(), 4 * bits.size(), cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_get_counters(cg_sim* s, uint64_t* attempts, uint64_t* proposals, uint64_t* iterations,
                               uint64_t* hops)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (attempts) *attempts = c.attempts;
    if (proposals) *proposals = c.proposals;
    if (iterations) *iterations = c.iterations;
    if (hops) *hops = c.hops;
    return CG_OK;
}

extern "C" int cg_enable_hop_log(cg_sim* s, uint64_t capacity, void* dev_buf, size_t bytes)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (s->own_log && s->d_log) { cudaFree(s->d_log); }
    s->d_log = nullptr; s->own_log = false; s->log_cap = 0; s->log_gap = false;
    if (capacity) {
        if (dev_buf) {
            if (bytes < 16 * capacity || ((uintptr_t)dev_buf & 7)) return CG_EINVAL;
            s->d_log = dev_buf;
        } else {
            CK(cudaMalloc(&s->d_log, 16 * capacity));
            s->own_log = true;
        }
        s->log_cap = capacity;
    }
    c.log_base = c.hops; c.log_a0 = c.attempts;
    CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_get_hops(cg_sim* s, uint64_t first, uint64_t count, uint64_t* attempt, uint32_t* i, uint32_t* j)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    const u64 have = std::min<u64>(c.hops - c.log_base, s->log_cap);
    if (first + count > have) return CG_EINVAL;
    if (!count) return CG_OK;
    const char* base = (const char*)s->d_log;
    if (attempt) CK(cudaMemcpyAsync(attempt, base + 8 * first, 8 * count, cudaMemcpyDeviceToHost, s->stream));
    if (i) CK(cudaMemcpyAsync(i, base + 8 * s->log_cap + 4 * first, 4 * count, cudaMemcpyDeviceToHost, s->stream));
    if (j) CK(cudaMemcpyAsync(j, base + 12 * s->log_cap + 4 * first, 4 * count, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_recompute_eps(cg_sim* s, double* max_abs_dev)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    cg_full_sum_eps<<<(s->N + 127) / 128, 128, 0, s->stream>>>(s->d_phi, s->d_nbits, s->d_tq, s->d_scratch,
                                                               s->L, s->lgL, s->pitch, s->N);
    CK(cudaMemsetAsync(s->d_red, 0, 8, s->stream));
    cg_max_abs_diff<<<std::max(1u, std::min(s->N / 256, 1024u)), 256, 0, s->stream>>>(s->d_scratch, s->d_eps[c.cur % CG_RING],
                                                                                     s->N, s->d_red);
    CK(cudaGetLastError());
    u64 bits = 0;
    CK(cudaMemcpyAsync(&bits, s->d_red, 8, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    double d; memcpy(&d, &bits, 8);
    if (max_abs_dev) *max_abs_dev = d;
    return CG_OK;
}

extern "C" int cg_apply_hops(cg_sim* s, uint64_t count, const uint32_t* i, const uint32_t* j, float* ms)
{
    if (!s || (count && (!i || !j))) return CG_EINVAL;
    if (ms) *ms = 0.f;
    if (!count) return CG_OK;
    for (u64 h = 0; h < count; ++h)
        if (i[h] >= s->N || j[h] >= s->N || i[h] == j[h]) return CG_EINVAL;
    u32* d_ij = nullptr;
    if (s->d_log) s->log_gap = true;
    CK(cudaMalloc(&d_ij, 8 * count));
    struct Free { void* p; ~Free() { cudaFree(p); } } fr{d_ij};
    CK(cudaMemcpyAsync(d_ij, i, 4 * count, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(d_ij + count, j, 4 * count, cudaMemcpyHostToDevice, s->stream));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    CgParams p = make_params(s, 0);
    // many small CTAs per SM (one block of 64 sites per warp; 128 threads measured best) keep enough
    // requests in flight to make the stand-alone update throughput-bound; larger lattices fall back to
    // one CTA per SM
    const u64 g1 = (s->N / 2 + 127) / 128;
    const int grid = (int)std::max<u64>(1, std::min<u64>((s->N / 2 + 511) / 512, (u64)s->num_sms));
    CK(cudaEventRecord(e0, s->stream));
    if (g1 <= (u64)s->num_sms * 12) cg_update_scripted<128, 1><<<(int)g1, 128, 0, s->stream>>>(p, d_ij, d_ij + count, count);
    else scripted_kernel(choose_rp(s->N / 2, grid, 512))<<<grid, 512, 0, s->stream>>>(p, d_ij, d_ij + count, count);
    CK(cudaEventRecord(e1, s->stream));
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(s->stream));
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (ms) *ms = t;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (c.bad_hops) {
        c.bad_hops = 0;
        CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        return CG_EINVAL;
    }
    return CG_OK;
}

extern "C" int cg_get_table_sizes(cg_sim* s, int64_t* K, int64_t* K_live)
{
    if (!s) return CG_EINVAL;
    if (K) *K = s->K;
    if (K_live) *K_live = s->Klive;
    return CG_OK;
}

extern "C" int cg_get_tables(cg_sim* s, int32_t* dy, int32_t* dx, double* cdf, double* invr_k, double* S, double* Gamma)
{
    if (!s) return CG_EINVAL;
    const size_t n = (size_t)s->Klive;
    if (dy) memcpy(dy, s->dy.data(), 4 * n);
    if (dx) memcpy(dx, s->dx.data(), 4 * n);
    if (cdf) memcpy(cdf, s->cdf.data(), 8 * n);
    if (invr_k) memcpy(invr_k, s->invr_k.data(), 8 * n);
    if (S) *S = s->S;
    if (Gamma) *Gamma = s->Gamma;
    return CG_OK;
}

extern "C" int cg_get_phi(cg_sim* s, double* phi)
{
    if (!s || !phi) return CG_EINVAL;
    CK(cudaMemcpyAsync(phi, s->d_phi, 8 * (size_t)s->N, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_set_launch(cg_sim* s, int n_ctas, int threads)
{
    if (!s || n_ctas < 0 || threads < 0) return CG_EINVAL;
    CK(cudaStreamSynchronize(s->stream));
    return choose_launch(s, n_ctas, threads);
}

extern "C" int cg_get_launch(cg_sim* s, int* n_ctas, int* threads, int* smem)
{
    if (!s) return CG_EINVAL;
    if (n_ctas) *n_ctas = s->n_ctas;
    if (threads) *threads = s->threads;
    if (smem) *smem = s->smem;
    return CG_OK;
}

extern "C" int cg_set_trace(cg_sim* s, void* dev_buf, size_t bytes, uint32_t iterations)
{
    if (!s) return CG_EINVAL;
    CK(cudaStreamSynchronize(s->stream));
    if (!dev_buf || !iterations) { s->d_trace = nullptr; s->trace_iters = 0; return CG_OK; }
#if !defined(CG_TRACE) && !defined(CG_TRACE_W) && !defined(CG_TRACE_T)
    return CG_EUNSUPPORTED;                   // the library was built without -DCG_TRACE
#endif
    if (((uintptr_t)dev_buf & 7) || bytes < (size_t)8 * 64 * CG_MAX_CTAS) return CG_EINVAL;
    s->d_trace = (u64*)dev_buf; s->trace_iters = iterations;
    return CG_OK;
}

extern "C" int cg_get_phase_cycles(cg_sim* s, uint64_t* total, uint64_t* wait, uint64_t* update,
                                   uint64_t* propose, int reset)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (total) *total = c.cyc_total;
    if (wait) *wait = c.cyc_wait;
    if (update) *update = c.cyc_update;
    if (propose) *propose = c.cyc_propose;
    if (reset) {
        c.cyc_total = c.cyc_wait = c.cyc_update = c.cyc_propose = 0;
        CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        CK(cudaStreamSynchronize(s->stream));
    }
    return CG_OK;
}

extern "C" int cg_bench_l2_rmw(size_t bytes, int reps, int trials, double* gbps)
{
    cg_sim* s = nullptr;
    if (!gbps || bytes < 4096 || (bytes & 15) || reps < 1 || trials < 1) return CG_EINVAL;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double2* buf = nullptr;
    CK(cudaMalloc(&buf, bytes));
    struct Free { void* p; ~Free() { cudaFree(p); } } fr{buf};
    CK(cudaMemset(buf, 0, bytes));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    const size_t n16 = bytes / 16;
    const int grid = (int)std::max<size_t>(1, std::min<size_t>((n16 + 511) / 512, (size_t)sms * 2));
    cg_l2_rmw<<<grid, 512>>>(buf, n16, 2);                 // warm-up
    float best = 1e30f;
    for (int t = 0; t < trials; ++t) {
        CK(cudaEventRecord(e0));
        cg_l2_rmw<<<grid, 512>>>(buf, n16, reps);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        best = std::min(best, ms);
    }
    CK(cudaGetLastError());
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *gbps = 2.0 * (double)bytes * (double)reps / ((double)best * 1e-3) / 1e9;
    return CG_OK;
}

extern "C" const char* cg_strerror(int code)
{
    switch (code) {
        case CG_OK: return "ok";
        case CG_EINVAL: return "invalid argument";
        case CG_ENOMEM: return "out of memory or workspace too small";
        case CG_ECUDA: return "CUDA error (see cg_last_error)";
        case CG_EUNSUPPORTED: return "problem not supported by the sm_100a path";
    }
    return "unknown error";
}

extern "C" const char* cg_last_error(cg_sim* s) { return s ? s->err.c_str() : ""; }

// ------------------------------------------------ observables --
// Read-only passes over device state, outside the hot loop: the Gaussian time increment of step 3c
// (PAPER.md:78), the density of states, the polarisation series and sigma0.

// Standard normal deviate of executed hop h (reading G19): Box-Muller of the Philox block
// counter = (h lo, h hi, 3, 0); u1 in (0,1], u2 in [0,1), 53 bits each.
__device__ __forceinline__ double normal_of_hop(u64 h, u32 seed_lo, u32 seed_hi)
{
    u32 w0, w1, w2, w3;
    philox4x32_10((u32)h, (u32)(h >> 32), 3u, 0u, seed_lo, seed_hi, w0, w1, w2, w3);
    const u64 a = (((u64)w0 << 32) | w1) >> 11, b = (((u64)w2 << 32) | w3) >> 11;
    const double u1 = (double)(a + 1) * 0x1p-53, u2 = (double)b * 0x1p-53;
    const double rad = sqrt(__dmul_rn(-2.0, log(u1)));
    const double ang = __dmul_rn(6.283185307179586476925286766559, u2);
    return __dmul_rn(rad, cos(ang));
}

__global__ void cg_normals(double* __restrict__ z, u64 first, u64 count, u32 seed_lo, u32 seed_hi)
{
    for (u64 k = blockIdx.x * (u64)blockDim.x + threadIdx.x; k < count; k += (u64)gridDim.x * blockDim.x)
        z[k] = normal_of_hop(first + k, seed_lo, seed_hi);
}

// Fixed-shape tree sum of a CTA's values (256 threads): the result depends on the launch shape only.
__device__ __forceinline__ double cta_sum_256(double v, double* sh)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = __dadd_rn(v, __shfl_down_sync(CG_FULL, v, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = threadIdx.x < 8 ? sh[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 4; o; o >>= 1) r = __dadd_rn(r, __shfl_down_sync(CG_FULL, r, o));
    }
    __syncthreads();
    return r;                               // valid in thread 0
}

// dt_h = m_h/Gamma + (sqrt(m_h)/Gamma) z_h, m_h from consecutive logged attempt indices;
// CTA c sums logged hops [c*chunk, (c+1)*chunk) in a fixed order.
__global__ void __launch_bounds__(256) cg_stoch_time_partial(const u64* __restrict__ log_a, u64 count, u64 a0,
                                                             u64 hop0, double Gamma, u32 seed_lo, u32 seed_hi,
                                                             u64 chunk, double* __restrict__ partial)
{
    __shared__ double sh[8];
    const u64 lo = blockIdx.x * chunk, hi = min(lo + chunk, count);
    double acc = 0.0;
    for (u64 h = lo + threadIdx.x; h < hi; h += 256) {
        const u64 prev = h ? log_a[h - 1] + 1 : a0;
        const double m = (double)(log_a[h] + 1 - prev);
        const double mean = __ddiv_rn(m, Gamma), sd = __ddiv_rn(sqrt(m), Gamma);
        acc = __dadd_rn(acc, __dadd_rn(mean, __dmul_rn(sd, normal_of_hop(hop0 + h, seed_lo, seed_hi))));
    }
    const double r = cta_sum_256(acc, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = r;
}

__global__ void __launch_bounds__(256) cg_sum_partials(const double* __restrict__ partial, u32 n, double* out)
{
    __shared__ double sh[8];
    double acc = 0.0;
    for (u32 k = threadIdx.x; k < n; k += 256) acc = __dadd_rn(acc, partial[k]);
    const double r = cta_sum_256(acc, sh);
    if (threadIdx.x == 0) *out = r;
}

// Density of states as bin counts: bin b = [lo + b*width, lo + (b+1)*width).
// CTA-private bins in shared memory when they fit (nsh = nbins), else global atomics (nsh = 0).
__global__ void __launch_bounds__(256) cg_dos(const double* __restrict__ eps, u32 N, double lo, double width,
                                              u32 nbins, u32 nsh, unsigned long long* __restrict__ hist /* nbins + 1 */)
{
    extern __shared__ u32 sh_bins[];
    for (u32 b = threadIdx.x; b < nsh; b += 256) sh_bins[b] = 0;
    __syncthreads();
    u32 outside = 0;
    for (u32 k = blockIdx.x * 256 + threadIdx.x; k < N; k += gridDim.x * 256) {
        const double x = floor(__ddiv_rn(__dsub_rn(eps[k], lo), width));
        if (x >= 0.0 && x < (double)nbins) {
            if (nsh) atomicAdd(&sh_bins[(u32)x], 1u);
            else atomicAdd(&hist[(u32)x], 1ull);
        } else ++outside;
    }
    outside = __reduce_add_sync(CG_FULL, outside);
    if ((threadIdx.x & 31) == 0 && outside) atomicAdd(&hist[nbins], (unsigned long long)outside);
    __syncthreads();
    for (u32 b = threadIdx.x; b < nsh; b += 256)
        if (sh_bins[b]) atomicAdd(&hist[b], (unsigned long long)sh_bins[b]);
}

// Polarisation series: P_h = sum of dx over logged hops 0..h, t_h = (a_h + 1)/Gamma.
#define CG_SCAN_ITEMS 8
#define CG_SCAN_CHUNK (256 * CG_SCAN_ITEMS)
__device__ __forceinline__ int hop_dx(u32 i, u32 j, int L)
{
    int d = ((int)(j & (u32)(L - 1)) - (int)(i & (u32)(L - 1))) & (L - 1);
    return d > L / 2 ? d - L : d;           // minimum image, tie -> +L/2 (G3)
}

__global__ void __launch_bounds__(256) cg_series_chunk_sums(const u32* __restrict__ li, const u32* __restrict__ lj,
                                                            u64 count, int L, long long* __restrict__ sums)
{
    __shared__ long long sh[8];
    const u64 base = blockIdx.x * (u64)CG_SCAN_CHUNK;
    long long acc = 0;
    for (int k = 0; k < CG_SCAN_ITEMS; ++k) {
        const u64 h = base + (u64)k * 256 + threadIdx.x;
        if (h < count) acc += hop_dx(li[h], lj[h], L);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) acc += __shfl_down_sync(CG_FULL, acc, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) { long long t = 0; for (int w = 0; w < 8; ++w) t += sh[w]; sums[blockIdx.x] = t; }
}

__global__ void cg_series_scan_sums(long long* sums, u32 n)       // exclusive scan, one CTA of 256 threads
{
    __shared__ long long sh[256];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (u32 base = 0; base < n; base += 256) {
        const u32 k = base + threadIdx.x;
        const long long v = k < n ? sums[k] : 0;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 256; o <<= 1) {
            const long long t = threadIdx.x >= (u32)o ? sh[threadIdx.x - o] : 0;
            __syncthreads();
            sh[threadIdx.x] += t;
            __syncthreads();
        }
        if (k < n) sums[k] = carry + sh[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += sh[255];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) cg_series_write(const u64* __restrict__ la, const u32* __restrict__ li,
                                                       const u32* __restrict__ lj, u64 first, u64 end, int L,
                                                       double Gamma, const long long* __restrict__ sums,
                                                       double* __restrict__ t, long long* __restrict__ P)
{
    __shared__ long long sh[8];
    const u64 h0 = blockIdx.x * (u64)CG_SCAN_CHUNK + (u64)threadIdx.x * CG_SCAN_ITEMS;   // 8 consecutive hops per thread
    long long v[CG_SCAN_ITEMS], run = 0;
#pragma unroll
    for (int k = 0; k < CG_SCAN_ITEMS; ++k) {
        const u64 h = h0 + k;
        run += h < end ? hop_dx(li[h], lj[h], L) : 0;
        v[k] = run;
    }
    long long inc = run;                                         // inclusive scan of the thread totals
    const u32 lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(CG_FULL, inc, o); if (lane >= (u32)o) inc += y; }
    if (lane == 31) sh[w] = inc;
    __syncthreads();
    long long off = sums[blockIdx.x] + inc - run;
    for (u32 k = 0; k < w; ++k) off += sh[k];
#pragma unroll
    for (int k = 0; k < CG_SCAN_ITEMS; ++k) {
        const u64 h = h0 + k;
        if (h >= first && h < end) {
            if (P) P[h - first] = off + v[k];
            if (t) t[h - first] = __ddiv_rn((double)(la[h] + 1), Gamma);
        }
    }
}

// Logged hops since the log was enabled; CG_EINVAL when the log is off or has overflowed (the observables
// over the log need every hop since the enabling point).
static int logged_hops(cg_sim* s, const CgCtl& c, u64* have)
{
    if (!s->d_log || !s->log_cap || s->log_gap) return CG_EINVAL;
    const u64 n = c.hops - c.log_base;
    if (n > s->log_cap) return CG_EINVAL;
    *have = n;
    return CG_OK;
}

struct DevTmp {             // scratch of one observable call, released on every return path
    void* p = nullptr;
    ~DevTmp() { if (p) cudaFree(p); }
};

extern "C" int cg_get_normals(cg_sim* s, uint64_t first_hop, uint64_t count, double* z)
{
    if (!s || (count && !z)) return CG_EINVAL;
    if (!count) return CG_OK;
    DevTmp tmp;
    CK(cudaMalloc(&tmp.p, 8 * count));
    const unsigned grid = (unsigned)std::min<u64>((count + 255) / 256, 148 * 8);
    cg_normals<<<grid, 256, 0, s->stream>>>((double*)tmp.p, first_hop, count, (u32)s->seed, (u32)(s->seed >> 32));
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(z, tmp.p, 8 * count, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_get_time_stochastic(cg_sim* s, double* t_tau0)
{
    if (!s || !t_tau0) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    u64 have = 0;
    if ((rc = logged_hops(s, c, &have)) != CG_OK) return rc;
    const double t0 = (double)c.log_a0 / s->Gamma;           // before the log: deterministic increment
    if (!have) { *t_tau0 = t0; return CG_OK; }
    const u64 chunk = 4096;
    const u32 nchunks = (u32)((have + chunk - 1) / chunk);
    DevTmp tmp;
    CK(cudaMalloc(&tmp.p, 8 * ((size_t)nchunks + 1)));
    double* partial = (double*)tmp.p;
    cg_stoch_time_partial<<<nchunks, 256, 0, s->stream>>>((const u64*)s->d_log, have, c.log_a0, c.log_base, s->Gamma,
                                                         (u32)s->seed, (u32)(s->seed >> 32), chunk, partial);
    cg_sum_partials<<<1, 256, 0, s->stream>>>(partial, nchunks, partial + nchunks);
    CK(cudaGetLastError());
    double sum = 0.0;
    CK(cudaMemcpyAsync(&sum, partial + nchunks, 8, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    *t_tau0 = t0 + sum;
    return CG_OK;
}

extern "C" int cg_get_dos(cg_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside)
{
    if (!s || !hist || !(width > 0.0) || nbins == 0 || nbins > (1u << 24)) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    DevTmp tmp;
    CK(cudaMalloc(&tmp.p, 8 * ((size_t)nbins + 1)));
    CK(cudaMemsetAsync(tmp.p, 0, 8 * ((size_t)nbins + 1), s->stream));
    const u32 nsh = nbins <= 8192 ? nbins : 0;               // 32 KB of CTA-private bins
    const unsigned grid = std::max(1u, std::min((s->N + 2047) / 2048, 148u * 4));
    cg_dos<<<grid, 256, 4 * (size_t)nsh, s->stream>>>(s->d_eps[c.cur % CG_RING], s->N, lo, width, nbins, nsh,
                                                      (unsigned long long*)tmp.p);
    CK(cudaGetLastError());
    std::vector<uint64_t> h((size_t)nbins + 1);
    CK(cudaMemcpyAsync(h.data(), tmp.p, 8 * h.size(), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    memcpy(hist, h.data(), 8 * (size_t)nbins);
    if (outside) *outside = h[nbins];
    return CG_OK;
}

extern "C" int cg_get_series(cg_sim* s, uint64_t first, uint64_t count, double* t, int64_t* P)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    u64 have = 0;
    if ((rc = logged_hops(s, c, &have)) != CG_OK) return rc;
    if (first + count > have) return CG_EINVAL;
    if (!count || (!t && !P)) return CG_OK;
    const u64 end = first + count;
    const u32 nchunks = (u32)((end + CG_SCAN_CHUNK - 1) / CG_SCAN_CHUNK);
    DevTmp tmp;
    const size_t off_t = align256(8 * (size_t)nchunks), off_P = off_t + align256(8 * count);
    CK(cudaMalloc(&tmp.p, off_P + 8 * count));
    long long* sums = (long long*)tmp.p;
    double* d_t = (double*)((char*)tmp.p + off_t);
    long long* d_P = (long long*)((char*)tmp.p + off_P);
    const u64* la = (const u64*)s->d_log;
    const u32* li = (const u32*)((const char*)s->d_log + 8 * s->log_cap);
    const u32* lj = (const u32*)((const char*)s->d_log + 12 * s->log_cap);
    cg_series_chunk_sums<<<nchunks, 256, 0, s->stream>>>(li, lj, end, s->L, sums);
    cg_series_scan_sums<<<1, 256, 0, s->stream>>>(sums, nchunks);
    cg_series_write<<<nchunks, 256, 0, s->stream>>>(la, li, lj, first, end, s->L, s->Gamma, sums, d_t, d_P);
    CK(cudaGetLastError());
    if (t) CK(cudaMemcpyAsync(t, d_t, 8 * count, cudaMemcpyDeviceToHost, s->stream));
    if (P) CK(cudaMemcpyAsync(P, d_P, 8 * count, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CG_OK;
}

extern "C" int cg_get_sigma0(cg_sim* s, double* sigma0)
{
    if (!s || !sigma0) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (s->E == 0.0 || c.attempts == 0) return CG_EINVAL;
    const double t = (double)c.attempts / s->Gamma;
    *sigma0 = (double)c.dP / (((double)s->N * s->E) * t);    // sigma0 = P/(N E t)
    return CG_OK;
}
