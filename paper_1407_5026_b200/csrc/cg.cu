// cg.cu — libcg.so: parallel-rejection kinetic Monte Carlo of the 2D Coulomb glass
// (Ferrero, Kolton, Palassini, arXiv 1407.5026) for NVIDIA B200 (sm_100a).
//
// The ABI is declared and documented in include/cg.h.  DESIGN.md explains the
// kernel design; the short version:
//   * one persistent cooperative kernel runs the whole propose -> select ->
//     apply -> update loop; there is ONE grid-wide exchange per
//     PR iteration, which carries both the lowest accepting label and the
//     "all local-energy slabs are written" guarantee;
//   * eps is double-buffered: after hop h every CTA writes eps_h for its own slab
//     into the other buffer while proposals read eps_{h-1} and add the pending
//     correction 1/r_lj - 1/r_li of hop h themselves (same single rounded add as
//     the update, so the values are bit-identical to the serial algorithm);
//   * occupations live as a bitmap in every CTA's shared memory, next to the live
//     part of the tower; 1/r comes from a quarter table in L2.
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

#define CG_SLOT_U64 32      // one exchange slot per CTA, 256-byte stride (own L2 slice), in u64 units
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
};

struct CgParams {           // kernel parameter block
    double* eps[2];         // double-buffered local energies, N each
    const double* tq;       // quarter table 1/r, (L/2+1) x (L/2+1)
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
    u32 seed_lo, seed_hi;
    double T, E;
    float inv_T;            // (float)(1/T), pre-test of the Metropolis factor only
    u64 n_hops;
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
__device__ __forceinline__ void fence_acquire_gpu() { asm volatile("fence.acquire.gpu;" ::: "memory"); }
// named barrier 1: the warps that wrote eps arrive, the publishing warp waits for them
__device__ __forceinline__ void bar1_arrive(int n) { asm volatile("bar.arrive 1, %0;" ::"r"(n) : "memory"); }
__device__ __forceinline__ void bar1_sync(int n) { asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory"); }

// 1/r between site (y,x) and site (yb,xb) under minimum image, from
// the quarter table; 0 on the diagonal.
__device__ __forceinline__ double invr_at(const double* __restrict__ tq, int pitch, int L,
                                          int y, int x, int yb, int xb)
{
    int dy = (y - yb) & (L - 1); dy = min(dy, L - dy);
    int dx = (x - xb) & (L - 1); dx = min(dx, L - dx);
    return __ldg(tq + dy * pitch + dx);
}

// Step 3b of the mixed PR algorithm: what hop i->j adds to eps at (y,x):
// 1/r_lj - 1/r_li (difference first, then ONE add by the caller).
__device__ __forceinline__ double hop_term(const double* __restrict__ tq, int pitch, int L,
                                           int y, int x, int yi, int xi, int yj, int xj)
{
    return __dsub_rn(invr_at(tq, pitch, L, y, x, yj, xj), invr_at(tq, pitch, L, y, x, yi, xi));
}

// The two terms of a pair of adjacent sites (y, x), (y, x+1), x even: both rows once.
__device__ __forceinline__ void hop_term2(const double* __restrict__ tq, int pitch, int L,
                                          int y, int x, int yi, int xi, int yj, int xj,
                                          double& c0, double& c1)
{
    int dyj = (y - yj) & (L - 1); dyj = min(dyj, L - dyj);
    int dyi = (y - yi) & (L - 1); dyi = min(dyi, L - dyi);
    const double* __restrict__ rj = tq + dyj * pitch;
    const double* __restrict__ ri = tq + dyi * pitch;
    int aj = (x - xj) & (L - 1), bj = (aj + 1) & (L - 1);
    int ai = (x - xi) & (L - 1), bi = (ai + 1) & (L - 1);
    aj = min(aj, L - aj); bj = min(bj, L - bj); ai = min(ai, L - ai); bi = min(bi, L - bi);
    const double j0 = __ldg(rj + aj), j1 = __ldg(rj + bj), i0 = __ldg(ri + ai), i1 = __ldg(ri + bi);
    c0 = __dsub_rn(j0, i0);
    c1 = __dsub_rn(j1, i1);
}

// eps slab of one CTA: pairs [pr0, pr1) of adjacent sites.  With RP > 0 thread t keeps pairs
// pr0 + t + k*THREADS (k < RP) in registers across hops and writes every new value through to
// global memory for the other CTAs' gathers; with RP == 0 the slab streams src -> dst.
template <int THREADS, int RP>
struct Slab {
    double2 e[RP > 0 ? RP : 1];

    __device__ __forceinline__ void load(const double* src, u32 pr0, u32 pr1)
    {
#pragma unroll
        for (int k = 0; k < RP; ++k) {
            const u32 pr = pr0 + threadIdx.x + k * THREADS;
            if (pr < pr1) e[k] = __ldcg(reinterpret_cast<const double2*>(src + 2 * pr));
        }
    }

    // dst = eps + (1/r_lj - 1/r_li) for every site l of the slab
    __device__ __forceinline__ void update(const CgParams& p, const double* src, double* dst,
                                           u32 pr0, u32 pr1, u32 hi, u32 hj)
    {
        const int L = p.L, lg = p.lgL, pitch = p.pitch;
        const int yi = hi >> lg, xi = hi & (L - 1), yj = hj >> lg, xj = hj & (L - 1);
        if (RP > 0) {
            double c0[RP > 0 ? RP : 1], c1[RP > 0 ? RP : 1];
#pragma unroll
            for (int k = 0; k < RP; ++k) {            // all table gathers first
                const u32 pr = pr0 + threadIdx.x + k * THREADS;
                if (pr < pr1) {
                    const u32 s = pr * 2;
                    hop_term2(p.tq, pitch, L, s >> lg, s & (L - 1), yi, xi, yj, xj, c0[k], c1[k]);
                }
            }
#pragma unroll
            for (int k = 0; k < RP; ++k) {
                const u32 pr = pr0 + threadIdx.x + k * THREADS;
                if (pr < pr1) {
                    e[k].x = __dadd_rn(e[k].x, c0[k]);
                    e[k].y = __dadd_rn(e[k].y, c1[k]);
                    __stcg(reinterpret_cast<double2*>(dst + 2 * pr), e[k]);
                }
            }
        } else {
            for (u32 pr = pr0 + threadIdx.x; pr < pr1; pr += THREADS) {
                const u32 s = pr * 2;
                const double2 v = __ldcg(reinterpret_cast<const double2*>(src + s));
                double a0, a1;
                hop_term2(p.tq, pitch, L, s >> lg, s & (L - 1), yi, xi, yj, xj, a0, a1);
                double2 o;
                o.x = __dadd_rn(v.x, a0);
                o.y = __dadd_rn(v.y, a1);
                __stcg(reinterpret_cast<double2*>(dst + s), o);
            }
        }
    }
};

// The persistent kernel: steps 1, 2, 3a-3c of the mixed PR algorithm.
template <int THREADS, int RP>
__global__ void __launch_bounds__(THREADS, 1) cg_pr_persistent(const CgParams p)
{
    constexpr int NW = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int KL = p.Klive;
    u64* s_cdfi = reinterpret_cast<u64*>(smem_raw);
    double* s_invr = reinterpret_cast<double*>(s_cdfi + KL);
    double* s_fld = s_invr + KL;
    int* s_disp = reinterpret_cast<int*>(s_fld + KL);
    u32* s_guide = reinterpret_cast<u32*>(s_disp + KL);
    u32* s_n = s_guide + CG_GUIDE;
    __shared__ u32 s_wlab[32], s_plab[32];
    __shared__ u64 s_wpay[32], s_ppay[32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 b = blockIdx.x, nb = gridDim.x;
    const int L = p.L, lg = p.lgL, pitch = p.pitch;
    const u32 N = p.N, M = p.M;

    for (int k = tid; k < KL; k += THREADS) {
        s_cdfi[k] = p.cdfi[k]; s_invr[k] = p.invr_k[k]; s_fld[k] = p.fld_k[k]; s_disp[k] = p.disp[k];
    }
    for (int k = tid; k < CG_GUIDE; k += THREADS) s_guide[k] = p.guide[k];
    for (u32 w = tid; w < (N + 31) / 32; w += THREADS) s_n[w] = p.nbits[w];

    // replicated, CTA-uniform control state
    u64 a0 = p.ctl->attempts, hops = p.ctl->hops, iters = p.ctl->iterations, props = p.ctl->proposals;
    long long dP = p.ctl->dP;
    u32 base = p.ctl->cur;
    u64 epoch = p.ctl->epoch;
    const u64 log_base = p.ctl->log_base;
    const u64 target = hops + p.n_hops;
    bool pending = false;                 // hop whose term readers must add to eps[base]
    u64 need_pub = 0;                     // epoch of the hop whose slabs must be complete before eps is read
    int pyi = 0, pxi = 0, pyj = 0, pxj = 0;
    u64 cyc_wait = 0, cyc_update = 0, cyc_propose = 0;
    const long long t_begin = clock64();

    const u32 per = (M + nb - 1) / nb;
    const u32 lab0 = min(M, b * per), lab1 = min(M, lab0 + per);
    const u32 pairs = N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    const u32 npw = min((u32)NW, (nb + 31) / 32);       // warps that poll the exchange slots
    u64* const my_slot = p.slots + (size_t)b * CG_SLOT_U64;

    Slab<THREADS, RP> slab;
    slab.load(p.eps[base], pr0, pr1);
    __syncthreads();

    while (hops < target) {
        const long long t0 = clock64();
        const double* __restrict__ erd = p.eps[base];
        // ---- steps 1-2: propose and test, state untouched
        u32 best = CG_NONE, bi = 0, bj = 0;
        for (u32 l = lab0 + tid; l < lab1; l += THREADS) {
            const u64 a = a0 + l;
            u32 w0, w1, w2, w3;
            philox4x32_10((u32)a, (u32)(a >> 32), 0u, 0u, p.seed_lo, p.seed_hi, w0, w1, w2, w3);
            const u32 i = __umulhi(w0, N);                                   // uniform site
            if (!((s_n[i >> 5] >> (i & 31)) & 1u)) continue;                 // n_i = 1 ?
            // tower sampling: smallest k with u_d < cdf_k, u_d = m 2^-43, as the
            // equivalent integer test m < cdfi_k; the guide brackets k from the leading bits of 1 - u_d
            const u64 m = ((u64)w1 << 11) | (u64)(w2 >> 21);
            const u64 t = (1ull << 43) - m;
            const int e = 63 - __clzll((long long)t);
            const u32 mant = (e >= 3 ? (u32)(t >> (e - 3)) : (u32)(t << (3 - e))) & 7u;
            const u32 g = s_guide[e * 8 + (int)mant];
            int lo = (int)(g & 0xFFFFu), hi = (int)(g >> 16);
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (m < s_cdfi[mid]) hi = mid; else lo = mid + 1;
            }
            const int d = s_disp[lo];
            const int dy = d >> 16, dx = (int)(short)(d & 0xFFFF);
            const int yi = i >> lg, xi = i & (L - 1);
            const int yj = (yi + dy) & (L - 1), xj = (xi + dx) & (L - 1);
            const u32 j = ((u32)yj << lg) | (u32)xj;
            if ((s_n[j >> 5] >> (j & 31)) & 1u) continue;                    // n_j = 0 ?
            double ei = ld_cg(erd + i), ej = ld_cg(erd + j);
            if (pending) {
                ei = __dadd_rn(ei, hop_term(p.tq, pitch, L, yi, xi, pyi, pxi, pyj, pxj));
                ej = __dadd_rn(ej, hop_term(p.tq, pitch, L, yj, xj, pyi, pxi, pyj, pxj));
            }
            // dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
            const double dE = __dsub_rn(__dsub_rn(__dsub_rn(ej, ei), s_invr[lo]), s_fld[lo]);
            bool acc = dE <= 0.0;
            if (!acc) {
                // Eq.(2): accept iff u_a < exp(-dE/T).  A float estimate with a 2^-10
                // guard band decides all but near-ties; those take the double-precision path, so the
                // decision is always that of the double comparison.
                const u32 uh = ((w2 & 0x1FFFFFu) << 11) | (w3 >> 21);        // top 32 of the 53 bits
                const float ul = (float)uh * 2.3283064365386963e-10f;        // u_a in [ul, ul + 2^-32)
                const float xf = (float)(-dE) * p.inv_T;
                const float pf = __expf(xf);
                int dec = 0;                                                 // 0 undecided, 1 accept, 2 reject
                if (ul > pf * 1.0009765625f) dec = 2;
                else if (xf > -60.f && ul + 4.6566128730773926e-10f < pf * 0.9990234375f) dec = 1;
                if (dec == 0) {
                    const double ua = (double)(((u64)(w2 & 0x1FFFFFu) << 32) | (u64)w3)
                                      * (1.0 / 9007199254740992.0);
                    acc = ua < exp(__ddiv_rn(-dE, p.T));
                } else acc = dec == 1;
            }
            if (acc) { best = l; bi = i; bj = j; break; }
        }
        const long long t1 = clock64();
        // ---- step 3: lowest accepting label: warp, CTA, grid
        {
            const u32 wmin = __reduce_min_sync(CG_FULL, best);
            const int src = __ffs(__ballot_sync(CG_FULL, best == wmin)) - 1;
            if (lane == src) { s_wlab[warp] = wmin; s_wpay[warp] = ((u64)bi << 32) | (u64)bj; }
        }
        __syncthreads();
        if (warp == 0) {
            const u32 lab = lane < NW ? s_wlab[lane] : CG_NONE;
            const u64 pay = lane < NW ? s_wpay[lane] : 0ull;
            const u32 gmin = __reduce_min_sync(CG_FULL, lab);
            const int src = __ffs(__ballot_sync(CG_FULL, lab == gmin)) - 1;
            if (lane == src) {
                if (nb > 1)
                    slot_store(my_slot, ((u64)(u32)epoch << 32) | gmin,
                               ((u64)((u32)epoch & 0xFFFFu) << 48) | ((pay >> 32) << 24) | (pay & 0xFFFFFFu));
                else { s_plab[0] = gmin; s_ppay[0] = pay; }
            }
        }
        if (nb > 1 && warp < npw) {
            // every slot is watched by one thread; the hop whose slabs the next gathers read must be
            // published too (pub word, written by each CTA after its eps stores are fenced)
            u32 plab = CG_NONE; u64 ppay = 0;
            const u32 e32 = (u32)epoch, e16 = (u32)epoch & 0xFFFFu;
            for (u32 c = tid; c < nb; c += THREADS) {
                const u64* sl = p.slots + (size_t)c * CG_SLOT_U64;
                u64 q0, q1;
                for (;;) {
                    slot_load(sl, q0, q1);
                    const u64 pb = ld_relaxed_u64(sl + 2);
                    if ((u32)(q0 >> 32) == e32 && (u32)(q1 >> 48) == e16 && pb >= need_pub) break;
                }
                if ((u32)q0 < plab) { plab = (u32)q0; ppay = ((q1 >> 24) & 0xFFFFFFull) << 32 | (q1 & 0xFFFFFFull); }
            }
            fence_acquire_gpu();
            const u32 wmin = __reduce_min_sync(CG_FULL, plab);
            const int src = __ffs(__ballot_sync(CG_FULL, plab == wmin)) - 1;
            if (lane == src) { s_plab[warp] = wmin; s_ppay[warp] = ppay; }
        }
        __syncthreads();
        u32 q, hi_, hj_;
        {
            const u32 lab = (u32)lane < npw ? s_plab[lane] : CG_NONE;
            const u64 pay = (u32)lane < npw ? s_ppay[lane] : 0ull;
            q = __reduce_min_sync(CG_FULL, lab);
            const int src = __ffs(__ballot_sync(CG_FULL, lab == q)) - 1;
            const u64 wp = __shfl_sync(CG_FULL, pay, src);
            hi_ = (u32)(wp >> 32); hj_ = (u32)wp;
        }
        const long long t2 = clock64();
        ++iters; props += M;
        cyc_propose += (u64)(t1 - t0); cyc_wait += (u64)(t2 - t1);
        if (q == CG_NONE) { a0 += M; ++epoch; continue; }   // whole window rejected: p += 1

        // ---- step 3a: execute the hop of label q; m = (p-1)M + q attempts used
        const u64 a_hop = a0 + q;
        a0 = a_hop + 1;
        const int yi = hi_ >> lg, xi = hi_ & (L - 1), yj = hj_ >> lg, xj = hj_ & (L - 1);
        int ddx = (xj - xi) & (L - 1); if (ddx > L / 2) ddx -= L;   // minimum image, tie -> +L/2
        dP += ddx;                                                   // step 3b: dP = dx
        if (tid == 0) {
            s_n[hi_ >> 5] &= ~(1u << (hi_ & 31));
            s_n[hj_ >> 5] |= (1u << (hj_ & 31));
            if (b == 0 && hops - log_base < p.log_cap) {
                const u64 h = hops - log_base;
                p.log_a[h] = a_hop; p.log_i[h] = hi_; p.log_j[h] = hj_;
            }
        }
        ++hops;
        __syncthreads();
        // ---- step 3b: local energies of my slab, into the other buffer
        if (pending) base ^= 1u;
        slab.update(p, p.eps[base], p.eps[base ^ 1u], pr0, pr1, hi_, hj_);
        pending = true; pyi = yi; pxi = xi; pyj = yj; pxj = xj;
        need_pub = epoch;
        if (nb > 1) {
            // publish "my slab of this hop is written" off the critical path: the last warp waits for
            // the others' stores (named barrier), fences them and releases the pub word
            if (warp == NW - 1) {
                bar1_sync(THREADS);
                if (lane == 0) st_release_u64(my_slot + 2, epoch);
            } else bar1_arrive(THREADS);
        }
        ++epoch;
        cyc_update += (u64)(clock64() - t2);
    }

    if (b == 0) {
        for (u32 w = tid; w < (N + 31) / 32; w += THREADS) p.nbits[w] = s_n[w];
        if (tid == 0) {
            CgCtl* c = p.ctl;
            c->attempts = a0; c->hops = hops; c->iterations = iters; c->proposals = props;
            c->dP = dP; c->cur = pending ? (base ^ 1u) : base; c->epoch = epoch;
            c->cyc_total += (u64)(clock64() - t_begin);
            c->cyc_wait += cyc_wait; c->cyc_update += cyc_update; c->cyc_propose += cyc_propose;
        }
    }
}

// Step a6 alone: scripted hops, update in place (no readers), one launch.
template <int THREADS, int RP>
__global__ void __launch_bounds__(THREADS, 1)
cg_update_scripted(const CgParams p, const u32* __restrict__ hop_i, const u32* __restrict__ hop_j, u64 count)
{
    const u32 b = blockIdx.x, nb = gridDim.x;
    const u32 pairs = p.N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    double* e = p.eps[p.ctl->cur];
    Slab<THREADS, RP> slab;
    slab.load(e, pr0, pr1);
    for (u64 h = 0; h < count; ++h)
        slab.update(p, e, e, pr0, pr1, __ldg(hop_i + h), __ldg(hop_j + h));
    if (b == 0 && threadIdx.x == 0) {       // occupations and dipole moment, in hop order
        long long dP = p.ctl->dP; u32 bad = 0;
        const int L = p.L;
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
    double* d_eps[2] = {nullptr, nullptr};
    double* d_scratch = nullptr; double* d_phi = nullptr;
    u32* d_nbits = nullptr; double* d_tq = nullptr;
    u64* d_cdfi = nullptr; double* d_invr_k = nullptr; double* d_fld_k = nullptr; int* d_disp = nullptr;
    u32* d_guide = nullptr;
    u64* d_slots = nullptr; CgCtl* d_ctl = nullptr; u64* d_red = nullptr;
    void* d_log = nullptr; bool own_log = false; u64 log_cap = 0;
    // launch shape
    int num_sms = 0, n_ctas = 0, threads = 0, smem = 0, rp = 0;
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

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static bool valid_L(int L, int* lg)
{
    if (L < 4 || L > 1024 || (L & (L - 1))) return false;
    int k = 0; while ((1 << k) < L) ++k;
    if (lg) *lg = k;
    return true;
}

struct WsLayout { size_t eps0, eps1, scratch, phi, nbits, tq, cdfi, invr_k, fld_k, disp, guide, slots, ctl, red, total; };
#define CG_SLOT_BYTES ((size_t)8 * CG_SLOT_U64 * CG_MAX_CTAS)

static WsLayout ws_layout(int L)
{
    const size_t N = (size_t)L * L, h = (size_t)L / 2 + 1;
    WsLayout w; size_t o = 0;
    w.eps0 = o; o += align256(8 * N);
    w.eps1 = o; o += align256(8 * N);
    w.scratch = o; o += align256(8 * N);
    w.phi = o; o += align256(8 * N);
    w.nbits = o; o += align256(N / 8 + 4);
    w.tq = o; o += align256(8 * h * h);
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
    p.eps[0] = s->d_eps[0]; p.eps[1] = s->d_eps[1];
    p.tq = s->d_tq; p.nbits = s->d_nbits;
    p.cdfi = s->d_cdfi; p.invr_k = s->d_invr_k; p.fld_k = s->d_fld_k; p.disp = s->d_disp;
    p.guide = s->d_guide;
    p.slots = s->d_slots; p.ctl = s->d_ctl;
    p.log_a = (u64*)s->d_log;
    p.log_i = s->d_log ? (u32*)((char*)s->d_log + 8 * s->log_cap) : nullptr;
    p.log_j = s->d_log ? (u32*)((char*)s->d_log + 12 * s->log_cap) : nullptr;
    p.log_cap = s->d_log ? s->log_cap : 0;
    p.L = s->L; p.lgL = s->lgL; p.pitch = s->pitch; p.Klive = (int)s->Klive;
    p.N = s->N; p.M = s->M;
    p.seed_lo = (u32)s->seed; p.seed_hi = (u32)(s->seed >> 32);
    p.T = s->T; p.E = s->E; p.inv_T = (float)(1.0 / s->T); p.n_hops = n_hops;
    return p;
}

typedef void (*persist_fn)(const CgParams);
typedef void (*scripted_fn)(const CgParams, const u32*, const u32*, u64);

// RP = eps pairs a thread keeps in registers (0: the slab streams through global memory)
template <int THREADS>
static persist_fn persistent_kernel_t(int rp)
{
    switch (rp) {
        case 0: return cg_pr_persistent<THREADS, 0>;
        case 1: return cg_pr_persistent<THREADS, 1>;
        case 2: return cg_pr_persistent<THREADS, 2>;
        case 4: return cg_pr_persistent<THREADS, 4>;
        case 8: return cg_pr_persistent<THREADS, 8>;
    }
    return nullptr;
}
static persist_fn persistent_kernel(int threads, int rp)
{
    switch (threads) {
        case 256: return persistent_kernel_t<256>(rp);
        case 512: return persistent_kernel_t<512>(rp);
        case 1024: return rp > 2 ? nullptr : persistent_kernel_t<1024>(rp);
    }
    return nullptr;
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
    const u64 need = (per_cta + threads - 1) / threads;
    const int cap = threads == 1024 ? 2 : 8;
    for (int rp = 1; rp <= cap; rp *= 2)
        if ((u64)rp >= need) return rp;
    return 0;
}

static int max_coresident(cg_sim* s, int threads, int rp, int* out)
{
    persist_fn f = persistent_kernel(threads, rp);
    if (!f) return CG_EINVAL;
    CK(cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem));
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)f, threads, s->smem));
    *out = std::min(per_sm * s->num_sms, CG_MAX_CTAS);
    return CG_OK;
}

static int choose_launch(cg_sim* s, int n_ctas, int threads)
{
    if (threads == 0) threads = 512;
    if (threads != 256 && threads != 512 && threads != 1024) return CG_EINVAL;
    const bool heuristic = n_ctas == 0;
    if (heuristic) {
        const u64 work = std::max<u64>(s->M, s->N / 2);
        n_ctas = (int)std::min<u64>((work + threads - 1) / threads, (u64)s->num_sms);
        n_ctas = std::max(1, n_ctas);
    }
    if (n_ctas < 1 || n_ctas > CG_MAX_CTAS) return CG_EINVAL;
    int rp = choose_rp(s->N / 2, n_ctas, threads);
    int cap = 0;
    int rc = max_coresident(s, threads, rp, &cap);
    if (rc != CG_OK) return rc;
    if (cap < 1) { s->err = "persistent kernel does not fit on an SM"; return CG_EUNSUPPORTED; }
    if (n_ctas > cap) {
        if (!heuristic) return CG_EINVAL;
        n_ctas = cap;
        rp = choose_rp(s->N / 2, n_ctas, threads);
        rc = max_coresident(s, threads, rp, &cap);
        if (rc != CG_OK) return rc;
        if (n_ctas > cap) return CG_EUNSUPPORTED;
    }
    if (n_ctas != s->n_ctas)   // slots of CTAs that no longer exist must not look published
        CK(cudaMemsetAsync(s->d_slots, 0, CG_SLOT_BYTES, s->stream));
    s->n_ctas = n_ctas; s->threads = threads; s->rp = rp;
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
    s->d_eps[0] = (double*)(base + w.eps0); s->d_eps[1] = (double*)(base + w.eps1);
    s->d_scratch = (double*)(base + w.scratch); s->d_phi = (double*)(base + w.phi);
    s->d_nbits = (u32*)(base + w.nbits); s->d_tq = (double*)(base + w.tq);
    s->d_cdfi = (u64*)(base + w.cdfi); s->d_invr_k = (double*)(base + w.invr_k);
    s->d_fld_k = (double*)(base + w.fld_k); s->d_guide = (u32*)(base + w.guide);
    s->d_disp = (int*)(base + w.disp); s->d_slots = (u64*)(base + w.slots);
    s->d_ctl = (CgCtl*)(base + w.ctl); s->d_red = (u64*)(base + w.red);

    std::vector<int> disp((size_t)s->Klive);
    for (int64_t k = 0; k < s->Klive; ++k) disp[k] = (s->dy[k] << 16) | (s->dx[k] & 0xFFFF);
    cudaStream_t st = s->stream;
    CK(cudaMemcpyAsync(s->d_tq, tq.data(), 8 * tq.size(), cudaMemcpyHostToDevice, st));
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
    if (s->own_ws && s->ws) cudaFree(s->ws);
    delete s;
}

extern "C" int cg_run(cg_sim* s, uint64_t n_hops)
{
    if (!s) return CG_EINVAL;
    if (n_hops == 0) return CG_OK;
    persist_fn f = persistent_kernel(s->threads, s->rp);
    if (!f) return CG_EINVAL;
    CgParams p = make_params(s, n_hops);
    void* args[] = {&p};
    CK(cudaLaunchCooperativeKernel((const void*)f, dim3(s->n_ctas), dim3(s->threads), args, (size_t)s->smem, s->stream));
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
    if (eps) CK(cudaMemcpyAsync(eps, s->d_eps[c.cur & 1], 8 * (size_t)s->N, cudaMemcpyDeviceToHost, s->stream));
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
    c.log_base = hops;
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
    s->d_log = nullptr; s->own_log = false; s->log_cap = 0;
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
    c.log_base = c.hops;
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
    cg_max_abs_diff<<<std::max(1u, std::min(s->N / 256, 1024u)), 256, 0, s->stream>>>(s->d_scratch, s->d_eps[c.cur & 1],
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
    CK(cudaMalloc(&d_ij, 8 * count));
    struct Free { void* p; ~Free() { cudaFree(p); } } fr{d_ij};
    CK(cudaMemcpyAsync(d_ij, i, 4 * count, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(d_ij + count, j, 4 * count, cudaMemcpyHostToDevice, s->stream));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    CgParams p = make_params(s, 0);
    const int grid = (int)std::max<u64>(1, std::min<u64>((s->N / 2 + 511) / 512, (u64)s->num_sms));
    scripted_fn uf = scripted_kernel(choose_rp(s->N / 2, grid, 512));
    CK(cudaEventRecord(e0, s->stream));
    uf<<<grid, 512, 0, s->stream>>>(p, d_ij, d_ij + count, count);
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
