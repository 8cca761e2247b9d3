// cg.cu — libcg.so: parallel-rejection kinetic Monte Carlo of the Coulomb glass
// (Ferrero, Kolton, Palassini, arXiv 1407.5026) for NVIDIA B200 (sm_100a).
//
// The ABI is declared and documented in include/cg.h.  DESIGN.md explains the
// kernel design; the short version:
//   * one persistent cooperative kernel runs the whole propose -> select ->
//     apply -> update loop, one CTA per SM, as a DATAFLOW between
//     warps instead of CTA-wide barriers: worker warps test proposals and update
//     their eps slab, a collector warp reduces the workers' results in label order
//     (stopping at the first accept), an exchange warp decides the iteration from
//     the CTAs' posts and publishes its outcome in a small ring of descriptors
//     (mbarrier full/empty pairs), a service warp publishes finished eps snapshots;
//     a worker may lag the exchange warp by up to CG_XR - 1 iterations, so only the
//     warps that hold the lowest labels sit on the critical path;
//   * the grid exchange is one-way most of the time: posts are scanned in label
//     order and the scan stops at the first accepting CTA; CTAs of one thread-block
//     cluster post into each other's shared memory (DSMEM), the others through L2;
//   * every thread owns the attempts a = g (mod P), keeps its proposal decoded and,
//     while theta_ij = 1, follows the two local energies it needs in registers by
//     adding every executed hop's term itself (the same rounded adds as the update);
//   * each CTA keeps its eps slab in registers and writes it through to a ring of
//     snapshot buffers every H hops (deferred update); readers only
//     touch a snapshot that every CTA has published and add the terms of the newer
//     hops in hop order, so no reader ever waits for a writer and every value is
//     bit-identical to the serial algorithm;
//   * occupations live as a bitmap in every CTA's shared memory (updated lazily,
//     readers replay the newest hops), next to the head of the tower (PAPER.md:71,
//     80) and its guide table; 1/r comes from an unfolded table in L2 indexed with
//     one subtraction and one mask (2D and 3D lattices share the code).
//   * a sim that fits ONE CTA (M <= 1024 labels, or up to 8 labels per thread on request; N <= 16384 sites)
//     runs in a kernel of its own (cg_pr_single, cg_pr_singlek): every thread a worker, eps, occupations and
//     the tower in shared memory, two CTA barriers per iteration; cg_run_many packs such sims one per SM.
// Nothing in this file is shared with oracle/ (the CPU reference).
#include "cg.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

typedef unsigned long long u64;
typedef unsigned int u32;

#define CG_NONE 0xFFFFFFFFu
#define CG_FULL 0xFFFFFFFFu
#define CG_MAX_CTAS 1024

// ------------------------------------------------------------------ device --

#ifndef CG_XR
#define CG_XR 4             // descriptor ring: the exchange warp may be this many iterations ahead of the slowest consumer
#endif
#ifndef CG_POLL_NS
#define CG_POLL_NS 0        // pause (ns) between two looks at shared memory of the polling role warps (0: none; 20-60 measured 1-2 % slower)
#endif
#ifndef CG_FRONT
#define CG_FRONT 2048u      // labels below this are "near the front" of the window
#endif
#define CG_PB 8             // publication barriers (snapshots a CTA's workers may be ahead of its service warp)
#define CG_HR 32            // hop ring: coded sites of the last CG_HR executed hops, for readers that catch up
#define CG_RING 12          // eps snapshot buffers (see "snapshots" in pr_persistent_body)
#define CG_SRING 32         // exchange slots per CTA (a CTA's posts may be this many iterations ahead of their slowest reader)
#define CG_SLOT_U64 128     // one 1 KiB block per CTA: the slot ring in the first half, the publication word after it
#define CG_PUB_U64 64
#define CG_GUIDE 352        // tower guide: (43 + 1) binades x 8 sub-buckets of t = 2^43 - m
#define CG_KS 2048          // head of the tower kept in shared memory (the rest, hardly ever drawn, stays in L2)
#define CG_MAX_CLUSTER 16
#define CG_MAX_SNAP 8       // largest snapshot interval H
#define CG_KMAX 8           // MULTI: most cached labels per thread
#define CG_XSLOT_BYTES 40   // MULTI: shared memory per extra label slot and thread

#define CG_F_HOP 1u         // descriptor flags: the iteration executed a hop
#define CG_F_LAST 2u        //   ... and it was the last one of this launch
#define CG_F_ABORT 4u       //   watchdog: give up

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
    u64 cyc_total, cyc_wait, cyc_update, cyc_propose;   // phase timers of CTA 0 (cg_get_phase_cycles)
    u64 pub_base;           // publication sequence number at the start of the next launch: CTA c stores
                            // pub_base + s into its pub word once its slab of snapshot s of a launch is
                            // written (never reset, so stale words of other launch shapes are always smaller)
    u64 log_a0;             // attempts consumed when the hop log was enabled (observables: m of the first logged hop)
    u32 abort;              // != 0: the watchdog of the persistent kernel fired (which wait: see cg.h)
    u32 pad;
    u64 cyc_warps;          // worker warps that contributed to cyc_wait/update/propose
    u64 cyc_x[6];           // exchange warps of all CTAs (cg_get_exchange_cycles): recycle, gate, own workers, scan, publish; CTAs
};

struct CgParams {           // kernel parameter block
    double* eps[CG_RING];   // ring of local-energy snapshot buffers, N each
    double* work;           // RP == 0 only: the CTAs' private working copy of eps
    const double* tf;       // unfolded table 1/r (see site_code)
    const double* tq;       // folded table 1/r, (Lz/2+1) x (L/2+1) x (L/2+1)
    u32* nbits;             // occupations, bit s of word s/32
    const u64* cdfi;        // live tower as integer thresholds: u_d < cdf_k  <=>  m < cdfi_k
    const double* invr_k;   // 1/r of displacement k (live part)
    const double* fld_k;    // E * dx of displacement k
    const u32* disp;        // coded displacement: site_code of ((dz mod L), (dy mod L), (dx mod L))
    const u32* guide;       // tower guide: klo | khi << 16 per bucket
    u64* slots;             // exchange slots, CG_SLOT_U64 per CTA
    CgCtl* ctl;
    u64* log_a; u32* log_i; u32* log_j; u64 log_cap;
    int L, lgL, Klive, Ksm; // Ksm = min(Klive, CG_KS) tower entries in shared memory
    u32 hi1, hi2, spare, mask;   // site coding (site_code)
    u32 N, M;
    u32 PL;                 // CACHED: threads per CTA that own attempts
    u32 seed_lo, seed_hi;
    double T, E;
    float inv_T;            // (float)(1/T), pre-test of the Metropolis factor only
    u32 n_hops;             // hops of this launch (cg_run splits longer runs)
    u32 snap_shift;         // snapshots every H = 1 << snap_shift hops
    u32 gate;               // G: hop h waits until every CTA has published the snapshot that covers hop h - G
    u32 cluster;            // CTAs per thread-block cluster (1: none)
    u32 K;                  // MULTI: cached labels per thread (attempts a, a + P, .., a + (K-1) P); else 1
    u32 xoff;               // MULTI: byte offset of the extra label slots in dynamic shared memory
    u64 watchdog_ns;        // a wait longer than this aborts the launch (0: never)
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

// ---- global memory: exchange slots and publication words ------------------------------
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
__device__ __forceinline__ u32 ld_relaxed_u32(const u32* p)
{
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
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

// ---- shared memory: 16-byte records, mbarriers, cluster (DSMEM) -----------------------
__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lds128(const void* p, u64& a, u64& b)
{
    asm volatile("ld.volatile.shared.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(smem_u32(p)) : "memory");
}
__device__ __forceinline__ void sts128(void* p, u64 a, u64 b)
{
    asm volatile("st.volatile.shared.v2.u64 [%0], {%1, %2};" ::"r"(smem_u32(p)), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ uint4 lds128u(const void* p)
{
    uint4 v;
    asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void sts128u(void* p, u32 x, u32 y, u32 z, u32 w)
{
    asm volatile("st.volatile.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(smem_u32(p)), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void sts64u(void* p, u32 x, u32 y)
{
    asm volatile("st.volatile.shared.v2.u32 [%0], {%1, %2};" ::"r"(smem_u32(p)), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ uint2 lds64u(const void* p)
{
    uint2 v;
    asm volatile("ld.volatile.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ u32 ld_acquire_cta(const u32* p)
{
    u32 v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void max_release_cta(u32* p, u32 v)
{
    asm volatile("red.release.cta.shared.max.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void mbar_init(u64* b, u32 count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* b)
{
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
// one try: the hardware suspends the warp until the phase completes or a short, system-defined time has passed
// (the variant with a suspend-time hint is compiled into a plain sleep of that length: never use it here)
__device__ __forceinline__ bool mbar_try(u64* b, u32 parity)
{
    u32 ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.b32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ bool mbar_test(u64* b, u32 parity)    // never suspends
{
    u32 ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.test_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.b32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_expect_tx(u64* b, u32 bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.release.cta.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// bulk asynchronous copy global -> shared memory (TMA engine, 16-byte granularity), completion counted on an mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, u32 bytes, u64* bar)
{
    asm volatile("cp.async.bulk.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_spin(u64* b, u32 parity)        // plain wait (kernels without a watchdog)
{
    while (!mbar_try(b, parity)) { }
    return true;
}
__device__ __forceinline__ u32 cluster_ctarank()
{
    u32 r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ u32 mapa_cluster(u32 smem_addr, u32 rank)
{
    u32 r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster128(u32 cluster_addr, u64 a, u64 b)
{
    asm volatile("st.shared::cluster.v2.u64 [%0], {%1, %2};" ::"r"(cluster_addr), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release;\n\tbarrier.cluster.wait.acquire;" ::: "memory");
}

// ---- site coding and the unfolded 1/r table ---------------------------------------------
// A site s = (z L + y) L + x (z = 0 in 2D) is coded as c(s) = (z 2L + y) 2L + x: one spare bit above
// the x and the y field.  With the spare bits set in the minuend, ONE subtraction and ONE mask give
// all periodic coordinate differences:
//   ((c(s) | spare) - c(t)) & mask = (((z_s - z_t) mod L) 2L + ((y_s - y_t) mod L)) 2L + ((x_s - x_t) mod L),
// which indexes tf[] = 1/r of that offset under minimum image, 0 at the origin; likewise
// (c(s) + c(d)) & mask is the code of the site s displaced by d.
struct Geo {
    u32 hi1, hi2, spare, mask, Lm1; int lg;
    __device__ __forceinline__ u32 code(u32 s) const { return s + (s & hi1) + ((s & hi2) << 1); }
    __device__ __forceinline__ u32 site(u32 c) const
    {
        return (c & Lm1) | ((c >> 1) & (Lm1 << lg)) | ((c >> 2) & (Lm1 << (2 * lg)));
    }
    __device__ __forceinline__ int dx(u32 si, u32 sj) const     // minimum image along the field, tie -> +L/2 (G3)
    {
        const int L = (int)Lm1 + 1;
        int d = ((int)(sj & Lm1) - (int)(si & Lm1)) & (int)Lm1;
        return d > L / 2 ? d - L : d;
    }
};

// Step 3b of the mixed PR algorithm: what hop i->j adds to eps at the site coded sc
// (spare bits set): 1/r_lj - 1/r_li (difference first, then ONE add by the caller).
__device__ __forceinline__ double hop_term(const double* __restrict__ tf, u32 mask, u32 sc, u32 ci, u32 cj)
{
    return __dsub_rn(__ldg(tf + ((sc - cj) & mask)), __ldg(tf + ((sc - ci) & mask)));
}

// eps slab of one CTA: sites [2 pr0, 2 pr1).  With RP > 0 warp w keeps the blocks of 64 consecutive
// sites number w, w + TW/32, ... (RP of them) in registers across hops - lane l holds sites l and
// 32 + l of a block, so that every load and store of the warp covers 256 contiguous bytes - and writes
// the values through to a snapshot buffer when asked to; with RP == 0 the slab lives in the CTA's part
// of a private working buffer in global memory (L2).
// issue() starts the table gathers of a hop, finish() adds (and stores): the caller puts independent
// work between the two.
template <int TW, int RP>
struct Slab {
    static constexpr int R = RP > 0 ? RP : 1;
    double ea[R], eb[R];
    double ja[R], ia[R], jb[R], ib[R];
    u32 sca[R], scb[R];                  // coded sites (spare bits set); sites outside the slab compute on code 0 and never store
    u32 valid;                           // bit 2k: site a of block k is mine, bit 2k+1: site b
    u32 hci, hcj;
    u32 tix;                             // index of this thread among the TW threads that hold the slab

    __device__ __forceinline__ u32 site_a(u32 pr0, int k) const
    {
        return 2u * (pr0 + (u32)k * TW + (tix & ~31u)) + (tix & 31u);
    }

    __device__ __forceinline__ void load(const double* src, double* work, u32 pr0, u32 pr1, const Geo& g, u32 t)
    {
        tix = t; valid = 0u;
        if (RP > 0) {
#pragma unroll
            for (int k = 0; k < RP; ++k) {
                const u32 sa = site_a(pr0, k), sb = sa + 32u;
                const bool va = sa < 2u * pr1, vb = sb < 2u * pr1;
                valid |= (va ? 1u : 0u) << (2 * k) | (vb ? 1u : 0u) << (2 * k + 1);
                sca[k] = va ? g.code(sa) | g.spare : g.spare;
                scb[k] = vb ? g.code(sb) | g.spare : g.spare;
                ea[k] = va ? __ldcg(src + sa) : 0.0;
                eb[k] = vb ? __ldcg(src + sb) : 0.0;
            }
        } else if (work != src) {
            for (u32 s = 2u * pr0 + tix; s < 2u * pr1; s += TW) __stcg(work + s, __ldcg(src + s));
        }
    }

    __device__ __forceinline__ void issue(const double* __restrict__ tf, u32 mask, u32 ci, u32 cj)
    {
        hci = ci; hcj = cj;
#pragma unroll
        for (int k = 0; k < RP; ++k) {
            ja[k] = __ldg(tf + ((sca[k] - cj) & mask)); ia[k] = __ldg(tf + ((sca[k] - ci) & mask));
            jb[k] = __ldg(tf + ((scb[k] - cj) & mask)); ib[k] = __ldg(tf + ((scb[k] - ci) & mask));
        }
    }

    // eps += 1/r_lj - 1/r_li for every site l of the slab; snap != nullptr: also stored there
    __device__ __forceinline__ void finish(const double* __restrict__ tf, u32 mask, const Geo& g, double* work,
                                           double* snap, u32 pr0, u32 pr1)
    {
        if (RP > 0) {
#pragma unroll
            for (int k = 0; k < RP; ++k) {
                ea[k] = __dadd_rn(ea[k], __dsub_rn(ja[k], ia[k]));
                eb[k] = __dadd_rn(eb[k], __dsub_rn(jb[k], ib[k]));
            }
            if (snap) flush(work, snap, pr0, pr1);
        } else {
            for (u32 s = 2u * pr0 + tix; s < 2u * pr1; s += TW) {
                const u32 c = g.code(s) | g.spare;
                const double tj = __ldg(tf + ((c - hcj) & mask)), ti = __ldg(tf + ((c - hci) & mask));
                const double v = __dadd_rn(__ldcg(work + s), __dsub_rn(tj, ti));
                __stcg(work + s, v);
                if (snap) __stcg(snap + s, v);
            }
        }
    }

    // the slab as it stands, into a snapshot buffer
    __device__ __forceinline__ void flush(const double* work, double* snap, u32 pr0, u32 pr1) const
    {
        if (RP > 0) {
#pragma unroll
            for (int k = 0; k < RP; ++k) {
                const u32 sa = site_a(pr0, k);
                if ((valid >> (2 * k)) & 1u) __stcg(snap + sa, ea[k]);
                if ((valid >> (2 * k + 1)) & 1u) __stcg(snap + sa + 32u, eb[k]);
            }
        } else {
            for (u32 s = 2u * pr0 + tix; s < 2u * pr1; s += TW) __stcg(snap + s, __ldcg(work + s));
        }
    }
};

struct Prop {               // one decoded attempt (a pure function of seed and attempt index)
    u32 ci, cj, k;          // coded sites (no spare bits) and tower index
    u32 uh, ul;             // the 53 acceptance bits: u_a = (uh 2^32 + ul) 2^-53, uh < 2^21
};

struct Tables {             // the tower: head in shared memory, the rest in global memory
    const u64* cdfi; const double* invr; const double* fld; const u32* disp; const u32* guide;
    const u64* g_cdfi; const double* g_invr; const double* g_fld; const u32* g_disp;
    u32 ks;
    __device__ __forceinline__ u64 cdf(u32 k) const { return k < ks ? cdfi[k] : __ldg(g_cdfi + k); }
    __device__ __forceinline__ double inv(u32 k) const { return k < ks ? invr[k] : __ldg(g_invr + k); }
    __device__ __forceinline__ double field(u32 k) const { return k < ks ? fld[k] : __ldg(g_fld + k); }
    __device__ __forceinline__ u32 dcode(u32 k) const { return k < ks ? disp[k] : __ldg(g_disp + k); }
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
        if (m < t.cdf(mid)) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// Attempt a -> proposal (reading G9): one Philox block, i = (w0 N) >> 32,
// displacement from 43 bits, acceptance uniform from the remaining 53.
// in two halves, for callers that spread the work: the random words (Philox), then the tower search
__device__ __forceinline__ Prop decode_words(const CgParams& p, const Geo& g, u64 a, u64& m)
{
    u32 w0, w1, w2, w3;
    philox4x32_10((u32)a, (u32)(a >> 32), 0u, 0u, p.seed_lo, p.seed_hi, w0, w1, w2, w3);
    Prop r;
    r.ci = g.code(__umulhi(w0, p.N));
    m = ((u64)w1 << 11) | (u64)(w2 >> 21);
    r.k = 0; r.cj = 0;
    r.uh = w2 & 0x1FFFFFu; r.ul = w3;
    return r;
}
__device__ __forceinline__ void decode_finish(const Tables& t, const Geo& g, Prop& r, u64 m)
{
    r.k = tower_search(t, m);
    r.cj = (r.ci + t.dcode(r.k)) & g.mask;
}
__device__ __forceinline__ Prop decode_attempt(const Tables& t, const CgParams& p, const Geo& g, u64 a)
{
    u64 m;
    Prop r = decode_words(p, g, a, m);
    decode_finish(t, g, r, m);
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

// Cached labels: does worker warp wr of the CTA at scan position kb hold a label of the window [0, M)?  Thread t of
// that CTA holds label (kb per + t - tr) mod P, tr = offset of the window start in the CTA at position 0; the labels of
// a warp are consecutive (mod P), and only the warp w0 = tr / 32 at position 0 can contain the wrap (label 0).
__device__ __forceinline__ bool warp_in_window(u32 kb, u32 tr, u32 wr, u32 w0, u32 per, u32 P, u32 M)
{
    if (kb == 0u && wr == w0) return true;
    u32 x = kb * per + 32u * wr + P - tr;       // < 2 P
    if (x >= P) x -= P;
    return x < M;
}

// What the exchange warp publishes about iteration e, in slot e % CG_XR of the descriptor ring.
struct __align__(16) Desc {
    u32 used;               // attempts consumed: q + 1, or M when the whole window was rejected
    u32 flags;              // CG_F_*
    u32 ci, cj;             // coded sites of the executed hop
    u32 c_first, t0r;       // CTA at scan position 0 of the NEXT iteration and the offset of its first label
    u32 hopno, pad;         // hops executed in this launch including this one
};

// The whole per-CTA communication area (static shared memory).
struct __align__(16) Comm {
    u64 full[CG_XR];        // mbarrier: descriptor e published (count 1)
    u64 empty[CG_XR];       // mbarrier: descriptor e consumed by every worker warp and the collector
    u64 pubbar[CG_PB];      // mbarrier: snapshot s stored by every worker warp
    Desc desc[CG_XR];
    u64 res[2 * CG_XR][32][2];  // results of the worker warps: (epoch << 32 | lowest accepting label, i << 32 | j);
                            // a worker is at most CG_XR iterations ahead of the collector, hence twice the ring
    u64 own[CG_XR][2];      // the CTA's result (collector -> exchange warp), same format
    u64 peer[CG_MAX_CLUSTER][CG_SRING][2];   // posts of the other CTAs of the cluster (DSMEM), slot format
    u32 hist[2 * CG_XR][4]; // the collector's copy of the last descriptors (flags, ci, cj, hopno), for the lazy bitmap
    u32 hops[CG_HR][2];     // coded sites (i, j) of executed hop h at h % CG_HR
    u32 ver;                // newest snapshot that every CTA has published (count within this launch)
    u32 nlow;               // hops up to this one are in the occupation bitmap
    u32 abort;              // the launch is being abandoned
};


struct Waiter {             // watchdog state of one waiting warp
    u64 t0; u32 spins;
    __device__ __forceinline__ void reset() { t0 = 0; spins = 0; }
};

// One step of a wait loop; true: give up (the launch is being abandoned or the watchdog fired).
__device__ __forceinline__ bool wait_poll(Waiter& w, const CgParams& p, Comm* cm, u32 code)
{
    if (((++w.spins) & 63u) != 0u) return false;
    if (*(volatile u32*)&cm->abort) return true;
    if ((w.spins & 1023u) != 0u) return false;
    if (ld_relaxed_u32(&p.ctl->abort)) { *(volatile u32*)&cm->abort = 1u; return true; }
    if (!p.watchdog_ns) return false;
    const u64 now = global_ns();
    if (!w.t0) { w.t0 = now; return false; }
    if (now - w.t0 > p.watchdog_ns) {
        atomicCAS(&p.ctl->abort, 0u, code);
        *(volatile u32*)&cm->abort = 1u;
        return true;
    }
    return false;
}

// wait for the phase with this parity of an mbarrier; false: gave up
__device__ __forceinline__ bool mbar_wait(u64* b, u32 parity, const CgParams& p, Comm* cm, u32 code)
{
    if (mbar_try(b, parity)) return true;
    Waiter w; w.reset();
    for (;;) {
        if (mbar_try(b, parity)) return true;
        if (wait_poll(w, p, cm, code)) return false;
    }
}

// The persistent kernel: steps 1, 2, 3a-3c of the mixed PR algorithm.
//
// CACHED: thread g of the grid owns the attempts a = g (mod P), P = nb * PL >= M, keeps its current and
// its next proposal decoded in registers (a proposal is a pure function of the seed and the attempt
// index) and, while theta_ij = 1, also the two local energies it needs, to which it adds the term of
// every executed hop itself; an iteration then only re-tests the proposal on the current state.
// Otherwise (M > P) CTA b evaluates labels [b per, (b+1) per) from scratch in every iteration, with the
// warps of the CTA in lock step (the occupation bitmap is then always current).
//
// Roles: warp 0 the service warp (S), warps 1 .. NW the workers, warp NW+1 the collector (C), NW+2 the exchange warp (X):
// the warp arbiter prefers high warp ids, and C and X sit on the path of every hand-over.  Iteration e ("exchange"), state S_e before it, outcome O_e:
//   worker:  test own label on S_e -> res[e][warp]; slab update of the hop of O_{e-1}; wait for O_e (mbarrier
//            full[e]); consume it (labels, occupations of the followed pair, followed energies); arrive empty[e]
//   C:       reduce res[e][*] in label order, stopping at the first accept -> own[e], the CTA's slot in L2
//            and the shared memory of its cluster peers; consume O_e
//   X:       gate on published snapshots; find the first accepting CTA in scan order (own[e], cluster
//            peers in shared memory, the others' slots in L2), stopping there; publish O_e; counters, log
//   S:       per snapshot: wait until every worker warp has stored its part (mbarrier pubbar), publish the
//            CTA's sequence number (st.release.gpu), find the newest snapshot published by ALL CTAs
//
// Snapshots (deferred update).  Snapshot s = eps after hop s H of this launch, in buffer
// (cur0 + s) % CG_RING; workers keep their slab current in registers after every hop but store it only
// then.  A proposal that starts to follow a pair of sites at hop h reads snapshot v = cm->ver (complete
// on every CTA) and adds the terms of hops v H + 1 .. h itself, in hop order - the same single rounded
// adds the update performs, so the values are bit-identical whatever v is.  X lets hop h through only
// when every CTA has published snapshot floor((h - G)/H): all workers of the grid are then within
// G + H - 1 hops of each other, a reader has at most that many terms to add (the hop ring holds them),
// and with CG_RING H > 2 G + 2 H - 2 no buffer is overwritten while it can still be read.
// Occupations: the bitmap lags (X applies the hop of O_{e - CG_XR} when it recycles that descriptor,
// i.e. when every warp has consumed it), so it is never ahead of a reader; a reader replays the hops
// after cm->nlow (set/clear in hop order is idempotent).
//
// Written as a device function of (parameters, CTA index, CTA count) so that one launch can also hold
// several sims side by side (cg_pr_persistent_many): nothing in it looks at blockIdx or gridDim.
template <int NW, int RP, bool CACHED, bool TIMED, bool MULTI = false>
__device__ __forceinline__ void pr_persistent_body(const CgParams& p, const u32 b, const u32 nb)
{
    static_assert(!MULTI || CACHED, "MULTI is a variant of the cached-label path");
    constexpr int TW = NW * 32;           // worker threads
    constexpr int THREADS = TW + 96;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int KS = p.Ksm;
    u64* s_cdfi = reinterpret_cast<u64*>(smem_raw);
    double* s_invr = reinterpret_cast<double*>(s_cdfi + KS);
    double* s_fld = s_invr + KS;
    u32* s_disp = reinterpret_cast<u32*>(s_fld + KS);
    u32* s_guide = s_disp + KS;
    u32* s_n = s_guide + CG_GUIDE;
    // MULTI: label slots 1 .. K-1 of every worker thread (slot 0 lives in registers), [physical slot][thread]
    const u32 KX = MULTI ? p.K - 1u : 0u;
    double* x_ei = reinterpret_cast<double*>(smem_raw + (MULTI ? p.xoff : 0u));
    double* x_ej = x_ei + KX * TW;
    u32* x_ci = reinterpret_cast<u32*>(x_ej + KX * TW);
    u32* x_cj = x_ci + KX * TW;
    u32* x_uh = x_cj + KX * TW;
    u32* x_ul = x_uh + KX * TW;
    u32* x_k = x_ul + KX * TW;
    u32* x_fl = x_k + KX * TW;            // bit 0: n_i, 1: n_j, 2: energies followed, 3: slot decoded
    __shared__ Comm cmem;
    Comm* const cm = &cmem;
    const Tables tb = {s_cdfi, s_invr, s_fld, s_disp, s_guide, p.cdfi, p.invr_k, p.fld_k, p.disp, (u32)KS};
    const Geo geo = {p.hi1, p.hi2, p.spare, p.mask, (u32)(p.L - 1), p.lgL};

    // warp 0 = service warp, warps 1 .. NW = workers, then the collector and the exchange warp: the warp arbiter prefers high
    // warp ids, and those two sit on the path of every hand-over between CTAs (measured: +2-3 % at configs 2 and 3, nothing
    // lost at config 5; the service warp mostly sleeps on its mbarrier)
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int role = wid == 0 ? 2 : wid == NW + 1 ? 0 : wid == NW + 2 ? 1 : 3, warp = wid - 1, tid = (int)threadIdx.x - 32;
    const int atid = threadIdx.x;         // index among all threads (set-up loops)
    const u32 N = p.N, M = p.M, mask = p.mask;
    const double* __restrict__ tf = p.tf;
    const u32 Hs = p.snap_shift, Hm = (1u << Hs) - 1u;

    for (int k = atid; k < KS; k += THREADS) {
        s_cdfi[k] = p.cdfi[k]; s_invr[k] = p.invr_k[k]; s_fld[k] = p.fld_k[k]; s_disp[k] = p.disp[k];
    }
    for (int k = atid; k < CG_GUIDE; k += THREADS) s_guide[k] = p.guide[k];
    for (u32 w = atid; w < (N + 31) / 32; w += THREADS) s_n[w] = p.nbits[w];
    // no record may look like one of this launch: tag them with the epoch before its first
    const u64 stale = (u64)((u32)p.ctl->epoch - 1u) << 32;
    for (u32 k = atid; k < sizeof(cm->res) / 8; k += THREADS) (&cm->res[0][0][0])[k] = stale;
    for (u32 k = atid; k < sizeof(cm->peer) / 8; k += THREADS) (&cm->peer[0][0][0])[k] = stale;
    if (atid == 0) {
        for (int k = 0; k < CG_XR; ++k) {
            mbar_init(&cm->full[k], 1); mbar_init(&cm->empty[k], NW + 1);
            cm->own[k][0] = stale; cm->own[k][1] = 0;
        }
        for (int k = 0; k < CG_PB; ++k) mbar_init(&cm->pubbar[k], NW);
        cm->ver = 0; cm->nlow = 0; cm->abort = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    const u64 a_start = p.ctl->attempts, pub_base = p.ctl->pub_base;
    const u32 cur0 = p.ctl->cur;          // snapshot 0 of this launch: the complete state it starts from
    const u32 e_start = (u32)p.ctl->epoch;
    const u32 n_hops = p.n_hops;
    const long long t_begin = clock64();

    // labels: CTA-blocked (scan order = CTA order) or, CACHED, cyclic in the global thread index
    const u32 per = CACHED ? p.PL : (M + nb - 1) / nb;
    const u32 lab0 = min(M, b * per), lab1 = min(M, lab0 + per);
    const u32 P = nb * per;               // CACHED: attempts a = g (mod P) belong to thread g
    u32 c_first = 0, t0r = 0;             // CACHED: CTA at scan position 0 and the offset of a0 in it
    if (CACHED) { const u32 g0 = (u32)(a_start % P); c_first = g0 / per; t0r = g0 - c_first * per; }
    const u32 csz = p.cluster;            // posts inside a cluster go through shared memory
    const u32 cl0 = csz > 1 ? b - cluster_ctarank() : b;        // first CTA of my cluster
    __syncthreads();
    if (csz > 1) cluster_sync_all();      // the peers' mbarriers and post areas exist before anybody writes to them

    const u32 pairs = N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    u64* const my_slot = p.slots + (size_t)b * CG_SLOT_U64;
    const u32 n_snaps = n_hops >> Hs;     // regular snapshots of this launch

    if (role == 2) {
        // ------------------------------------------------------------------ service warp ----
        for (u32 s = 1; s <= n_snaps; ++s) {
            if (!mbar_wait(&cm->pubbar[(s - 1) % CG_PB], ((s - 1) / CG_PB) & 1u, p, cm, 1u)) break;
            if (nb == 1) { if (lane == 0) max_release_cta(&cm->ver, s); continue; }
            if (lane == 0) st_release_u64(my_slot + CG_PUB_U64, pub_base + s);
            u64 vmin = ~0ull;
            for (u32 c0 = lane; c0 < nb; c0 += 32 * 8) {                // eight independent loads in flight
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
            if (lane == 0 && vmin > pub_base) max_release_cta(&cm->ver, (u32)(vmin - pub_base));    // stale words are smaller
        }
    } else if (role == 0) {
        // ---------------------------------------------------------------- collector warp ----
        // The CTA's lowest accepting label of every iteration (step 3), found in label order:
        // lane r looks at the r-th warp in that order.  In scan order every worker warp holds lower labels
        // than the next one, except that (CACHED) at scan position 0 the threads below the first label of
        // the window hold its END ("tail" labels >= tail0): those rank after every other label.
        u32 cf = c_first, tr = t0r;
        Waiter wd;
        u32 c_app = 0;                    // descriptors below this one are in the occupation bitmap
        // the hop of descriptor x goes into the bitmap (every warp has consumed it; this warp is the only writer of the
        // bitmap, and volatile stores of one thread stay in order)
        auto apply = [&](u32 x) {
            const uint4 hx = lds128u(&cm->hist[x % (2 * CG_XR)][0]);
            if (lane == 0 && (hx.x & CG_F_HOP)) {
                const u32 si = geo.site(hx.y), sj = geo.site(hx.z);
                volatile u32* w = s_n;
                w[si >> 5] &= ~(1u << (si & 31));
                w[sj >> 5] |= 1u << (sj & 31);
                *(volatile u32*)&cm->nlow = hx.w;
            }
        };
        u32 e_end = 0;
        for (u32 e = 0;; ++e) {
            const u32 xs = e % CG_XR, e32 = e_start + e;
            const u32 kb = b >= cf ? b - cf : b + nb - cf;
            // head labels of the CTA at position kb: [kb per - tr, (kb+1) per - tr); anything above (the tail at
            // position 0; MULTI: the labels of slots 1 .. K-1) ranks after every head label of the grid
            const u32 tail0 = CACHED ? (kb + 1u) * per - tr : CG_NONE;
            const u32 w0 = (CACHED && kb == 0) ? tr >> 5 : 0u;
            u32 wr = w0 + (u32)lane; if (wr >= (u32)NW) wr -= NW;
            // CACHED: a warp all of whose labels lie beyond the window (M < P) reports nothing anybody needs
            const bool mine = lane < NW && (!CACHED || warp_in_window(kb, tr, wr, w0, per, P, M));
            bool ready = !mine; u32 l = CG_NONE, tl = CG_NONE; u64 pay = 0;
            u32 gmin = CG_NONE; u64 gpay = 0;
            wd.reset();
            bool quit = false;
            for (;;) {
                if (!ready) {
                    u64 q0, q1;
                    lds128(&cm->res[e % (2 * CG_XR)][wr][0], q0, q1);
                    if ((u32)(q0 >> 32) == e32) {
                        ready = true; pay = q1;
                        const u32 v = (u32)q0;
                        if (v != CG_NONE && v >= tail0) tl = v; else l = v;
                    }
                }
                const u32 racc = __ballot_sync(CG_FULL, ready && l != CG_NONE);
                const u32 rnot = __ballot_sync(CG_FULL, !ready);
                const int fa = racc ? __ffs(racc) - 1 : 32, fn = rnot ? __ffs(rnot) - 1 : 32;
                if (CACHED && fa < fn) {                        // first accept in label order, everything before it rejected
                    gmin = __shfl_sync(CG_FULL, l, fa); gpay = __shfl_sync(CG_FULL, pay, fa);
                    break;
                }
                if (!rnot) {                                    // every warp is in (lock step, not CACHED: always waited for)
                    const u32 hm = __reduce_min_sync(CG_FULL, l);
                    const u32 tm = hm != CG_NONE ? hm : __reduce_min_sync(CG_FULL, tl);    // no head accept: lowest tail accept
                    if (tm != CG_NONE) {
                        const int src = __ffs(__ballot_sync(CG_FULL, (hm != CG_NONE ? l : tl) == tm)) - 1;
                        gmin = tm; gpay = __shfl_sync(CG_FULL, pay, src);
                    }
                    break;
                }
                if (wait_poll(wd, p, cm, 2u)) { quit = true; break; }
                if (CG_POLL_NS > 0) __nanosleep(CG_POLL_NS);
            }
            if (quit) break;
            // post: own[] for the exchange warp, the slot in L2 for the other CTAs, the peers' shared memory
            const u64 s0 = ((u64)e32 << 32) | gmin;
            if (lane == 0) sts128(&cm->own[xs][0], s0, gpay);
            if (nb > 1) {
                const u32 ring = e32 & (CG_SRING - 1u);
                const u64 s1 = ((u64)(e32 & 0xFFFFu) << 48) | ((gpay >> 32) << 24) | (gpay & 0xFFFFFFu);
                if (csz > 1 && (u32)lane < csz && cl0 + (u32)lane != b) {
                    const u32 ra = mapa_cluster(smem_u32(&cm->peer[b - cl0][ring][0]), (u32)lane);
                    st_cluster128(ra, s0, s1);
                }
                if (lane == 0) slot_store(my_slot + 2u * ring, s0, s1);
            }
            // consume O_e
            if (!mbar_wait(&cm->full[xs], (e / CG_XR) & 1u, p, cm, 3u)) break;
            const uint4 d0 = lds128u(&cm->desc[xs]);
            const uint4 d1 = lds128u(&cm->desc[xs].c_first);
            if (CACHED) {
                // the lazy occupation bitmap: descriptors that every warp has consumed (their empty phase is complete;
                // never more than one phase ahead of this test, because this warp is one of the consumers)
                if (lane == 0) sts128u(&cm->hist[e % (2 * CG_XR)][0], d0.y, d0.z, d0.w, d1.z);
                __syncwarp();
                while (c_app < e && mbar_test(&cm->empty[c_app % CG_XR], (c_app / CG_XR) & 1u)) { apply(c_app); ++c_app; }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&cm->empty[xs]);
            e_end = e + 1u;
            if (d0.y & (CG_F_LAST | CG_F_ABORT)) break;
            cf = d1.x; tr = d1.y;
        }
        if (!*(volatile u32*)&cm->abort) {
            // end of the launch: the remaining hops go into the bitmap once every warp is done with it
            asm volatile("bar.sync 1, %0;" ::"r"(THREADS) : "memory");
            if (CACHED) for (; c_app < e_end; ++c_app) apply(c_app);
            __syncwarp();
            asm volatile("bar.sync 2, %0;" ::"r"(THREADS) : "memory");
            if (csz > 1) cluster_sync_all();
        }
        return;

    } else if (role == 1) {
        // ----------------------------------------------------------------- exchange warp ----
        const u64 log_base = p.ctl->log_base, hops_start = p.ctl->hops;
        u64 used_sum = 0;                 // attempts consumed in this launch
        long long dP = 0;
        u32 e = 0, hc = 0;                // iterations (mod 2^32: ring positions and epoch tags only) and hops decided in this launch
        u64 its = 0;                      // iterations of this launch (a cold system runs many more iterations than hops)
        u32 ver = 0;                      // newest snapshot known to be published by every CTA
        Waiter wd;
        bool quit = false;
        u64 tx[5] = {0, 0, 0, 0, 0};
        long long xt = TIMED ? clock64() : 0;
        auto stamp = [&](int k) { if (TIMED) { const long long now = clock64(); tx[k] += (u64)(now - xt); xt = now; } };
        while (hc < n_hops) {
            const u32 xs = e % CG_XR, e32 = e_start + e;
            // (1) recycle the descriptor slot: every consumer is past iteration e - CG_XR
            if (CACHED && e >= CG_XR && !mbar_wait(&cm->empty[xs], ((e - CG_XR) / CG_XR) & 1u, p, cm, 4u)) { quit = true; break; }
            stamp(0);
            // (2) gate: every CTA has published the snapshot that covers hop hc + 1 - G
            if (nb > 1 && hc + 1u > p.gate) {
                const u32 need = (hc + 1u - p.gate) >> Hs;
                if (ver < need) ver = max(ver, *(volatile u32*)&cm->ver);
                if (ver < need) {
                    const u64 want = pub_base + need;
                    wd.reset();
                    for (;;) {
                        bool ok = true;
                        for (u32 c0 = lane; c0 < nb; c0 += 32 * 8) {
                            u64 v[8];
#pragma unroll
                            for (int k = 0; k < 8; ++k) {
                                const u32 c = c0 + 32 * k;
                                v[k] = c < nb ? ld_relaxed_u64(p.slots + (size_t)c * CG_SLOT_U64 + CG_PUB_U64) : ~0ull;
                            }
#pragma unroll
                            for (int k = 0; k < 8; ++k) ok = ok && v[k] >= want;
                        }
                        if (__all_sync(CG_FULL, ok)) break;
                        wd.spins |= 63u;
                        if (wait_poll(wd, p, cm, 5u)) { quit = true; break; }
                    }
                    if (quit) break;
                    fence_acquire_gpu();
                    ver = need;
                    if (lane == 0) max_release_cta(&cm->ver, need);
                }
            }
            // (3) the first accepting CTA in scan order (step 3).  Position 0 holds the start of
            // the window; a window of scan positions is polled at a time, starting narrow (the winner is nearly
            // always at the first positions), and polling stops at the first accept: posts of later CTAs are
            // never waited for, and the CTA at position 0, when it accepts, waits for nobody.
            stamp(1);
            const u32 kb = b >= c_first ? b - c_first : b + nb - c_first;
            const u32 tail0 = CACHED ? per - t0r : CG_NONE;
            const u32 ring = e32 & (CG_SRING - 1u), e16 = e32 & 0xFFFFu;
            u32 q = CG_NONE; u64 wp = 0;
            u32 tlab = CG_NONE; u64 tpay = 0;                          // lowest late accept among the positions of this lane
            // positions that hold labels of the window (all of them when it wraps around to position 0)
            const u32 npos = CACHED ? min(nb, (t0r + M + per - 1u) / per) : nb;
            u32 lo = 0, hi = min(npos, 4u);
            wd.reset();
            if (CACHED && kb == 0) {
                // My own workers hold the start of the window: their results, read directly in label order (the
                // collector does the same for the other CTAs' sake, but its hand-over would be one more hop on the path).
                // A head accept of mine decides the iteration; otherwise the scan below goes on from my own post.
                const u32 w0 = t0r >> 5;
                u32 wr = w0 + (u32)lane; if (wr >= (u32)NW) wr -= NW;
                bool ready = lane >= NW || !warp_in_window(0u, t0r, wr, w0, per, P, M); u32 l = CG_NONE; u64 pay = 0;
                for (;;) {
                    if (!ready) {
                        u64 q0, q1;
                        lds128(&cm->res[e % (2 * CG_XR)][wr][0], q0, q1);
                        if ((u32)(q0 >> 32) == e32) { ready = true; pay = q1; const u32 v = (u32)q0; if (v < tail0) l = v; }
                    }
                    const u32 racc = __ballot_sync(CG_FULL, ready && l != CG_NONE);
                    const u32 rnot = __ballot_sync(CG_FULL, !ready);
                    const int fa = racc ? __ffs(racc) - 1 : 32, fn = rnot ? __ffs(rnot) - 1 : 32;
                    if (fa < fn) { q = __shfl_sync(CG_FULL, l, fa); wp = __shfl_sync(CG_FULL, pay, fa); lo = npos; break; }
                    if (!rnot) break;                   // no head accept here: the general scan (my tail labels come from own[])
                    if (wait_poll(wd, p, cm, 6u)) { quit = true; break; }
                }
                if (quit) break;
            }
            stamp(2);
            while (lo < npos) {
                const u32 k = lo + (u32)lane;
                const bool mine = k < hi;
                u32 c = c_first + k; if (c >= nb) c -= nb;
                const bool local = mine && k != kb && csz > 1 && c - cl0 < csz;
                const u32 hb = CACHED ? (k + 1u) * per - t0r : CG_NONE;     // head labels of position k lie below this
                bool ready = !mine; u32 l = CG_NONE; u64 pay = 0;
                bool found = false;
                // Positions behind my own are looked at only once my own result is in and rejects: while it is awaited, the
                // loop then touches shared memory only (as soon as the posts of the positions before mine have arrived) and
                // notices it within a few tens of cycles instead of one L2 round trip of a poll nobody needs
                const bool own_here = kb != 0u && kb >= lo && kb < hi;
                bool hold = mine && own_here && k > kb;
                for (;;) {
                    if (!ready && !hold) {
                        u64 q0, q1;
                        if (k == kb) {
                            lds128(&cm->own[xs][0], q0, q1);
                            if ((u32)(q0 >> 32) == e32) { ready = true; l = (u32)q0; pay = q1; }
                        } else {
                            if (local) lds128(&cm->peer[c - cl0][ring][0], q0, q1);
                            else slot_load(p.slots + (size_t)c * CG_SLOT_U64 + 2u * ring, q0, q1);
                            if ((u32)(q0 >> 32) == e32 && (u32)(q1 >> 48) == e16) {
                                ready = true; l = (u32)q0;
                                pay = ((q1 >> 24) & 0xFFFFFFull) << 32 | (q1 & 0xFFFFFFull);
                            }
                        }
                        if (ready && l != CG_NONE && l >= hb) { if (l < tlab) { tlab = l; tpay = pay; } l = CG_NONE; }
                    }
                    const u32 racc = __ballot_sync(CG_FULL, ready && l != CG_NONE);
                    const u32 rnot = __ballot_sync(CG_FULL, !ready);
                    const int fa = racc ? __ffs(racc) - 1 : 32, fn = rnot ? __ffs(rnot) - 1 : 32;
                    if (fa < fn) {                      // first accepting position, everything before it rejected
                        q = __shfl_sync(CG_FULL, l, fa); wp = __shfl_sync(CG_FULL, pay, fa);
                        found = true;
                        break;
                    }
                    if (!rnot) break;                   // whole window rejected: widen
                    if (own_here && !((rnot | racc) >> (kb - lo) & 1u)) hold = false;      // my own result is in and rejects
                    if (kb != 0 || lo != 0) wd.spins |= 63u;      // polls through L2 are slow: look at the clock more often
                    else if (CG_POLL_NS > 0) __nanosleep(CG_POLL_NS);                 // shared memory only: leave the issue slots to the workers
                    if (wait_poll(wd, p, cm, 6u)) { quit = true; break; }
                }
                if (quit || found) break;
                lo = hi; hi = min(npos, lo + 32u);
            }
            if (quit) break;
            stamp(3);
            if (q == CG_NONE) {               // no head label accepted: the lowest of the late ones (labels are distinct)
                const u32 tmin = __reduce_min_sync(CG_FULL, tlab);
                if (tmin != CG_NONE) {
                    const int src = __ffs(__ballot_sync(CG_FULL, tlab == tmin)) - 1;
                    q = tmin; wp = __shfl_sync(CG_FULL, tpay, src);
                }
            }
            // lock step (not CACHED): every warp of this CTA has finished its tests of this iteration before the
            // bitmap changes
            if (!CACHED) {
                wd.reset();
                for (;;) {
                    u64 q0, q1;
                    lds128(&cm->own[xs][0], q0, q1);
                    if ((u32)(q0 >> 32) == e32) break;
                    if (wait_poll(wd, p, cm, 7u)) { quit = true; break; }
                }
                if (quit) break;
                if (e >= CG_XR && !mbar_wait(&cm->empty[xs], ((e - CG_XR) / CG_XR) & 1u, p, cm, 4u)) { quit = true; break; }
            }
            // (4) publish O_e: attempts consumed (m = (p-1)M + q per executed hop), the hop
            // (step 3a)
            const u32 used = q == CG_NONE ? M : q + 1;
            const u32 ci = (u32)(wp >> 32), cj = (u32)wp;               // coded sites
            const bool hop = q != CG_NONE;
            if (CACHED) {
                if (t0r + used < per) t0r += used;
                else {
                    u32 g0 = c_first * per + t0r + (MULTI ? used % P : used); if (g0 >= P) g0 -= P;      // used <= M (<= P unless MULTI)
                    c_first = g0 / per; t0r = g0 - c_first * per;
                }
            }
            if (hop) ++hc;
            const u32 flags = (hop ? CG_F_HOP : 0u) | (hc >= n_hops ? CG_F_LAST : 0u);
            if (lane == 0) {
                if (hop) sts64u(&cm->hops[hc % CG_HR][0], ci, cj);
                Desc* d = &cm->desc[xs];
                sts128u(&d->c_first, c_first, t0r, hc, 0u);
                sts128u(&d->used, used, flags, ci, cj);
                if (!CACHED && hop) {         // lock step: the bitmap is always current
                    const u32 si = geo.site(ci), sj = geo.site(cj);
                    volatile u32* w = s_n;
                    w[si >> 5] &= ~(1u << (si & 31));
                    w[sj >> 5] |= 1u << (sj & 31);
                    *(volatile u32*)&cm->nlow = hc;
                }
                mbar_arrive(&cm->full[xs]);   // release: the stores above are visible to whoever sees the phase complete
            }
            // (5) the bookkeeping, off the critical path
            used_sum += used;
            ++e; ++its;
            if (hop) {
                const u32 hi_ = geo.site(ci), hj_ = geo.site(cj);
                dP += geo.dx(hi_, hj_);                                  // step 3b: dP = dx
                const u64 h = hops_start + hc - 1u - log_base;
                if (lane == 0 && b == 0 && h < p.log_cap) {
                    p.log_a[h] = a_start + used_sum - 1; p.log_i[h] = hi_; p.log_j[h] = hj_;
                }
            }
            stamp(4);
        }
        if (quit) {                       // let the consumers of this CTA go (they see the abort flag in their waits)
            if (lane == 0) *(volatile u32*)&cm->abort = 1u;
            return;
        }
        asm volatile("bar.sync 1, %0;" ::"r"(THREADS) : "memory");
        if (b == 0 && lane == 0) {
            CgCtl* c = p.ctl;
            const u32 ns = n_snaps + ((n_hops & Hm) ? 1u : 0u);
            c->attempts = a_start + used_sum; c->hops = hops_start + hc;
            c->iterations += its; c->proposals += (u64)M * its;
            c->dP += dP; c->cur = (cur0 + ns) % CG_RING; c->epoch += its;
            c->pub_base = pub_base + ns;
            c->cyc_total += (u64)(clock64() - t_begin);
        }
        if (TIMED && lane == 0) {
            for (int k = 0; k < 5; ++k) atomicAdd(&p.ctl->cyc_x[k], tx[k]);
            atomicAdd(&p.ctl->cyc_x[5], 1ull);
        }
        __syncwarp();
        asm volatile("bar.sync 2, %0;" ::"r"(THREADS) : "memory");
        if (b == 0) for (u32 w = lane; w < (N + 31) / 32; w += 32) p.nbits[w] = s_n[w];
        if (csz > 1) cluster_sync_all();  // no CTA leaves while a peer may still post into its shared memory
        return;
    } else {
        // ------------------------------------------------------------------ worker warps ----
        // CACHED per-thread state: label of my attempt relative to the window start, the decoded proposal and
        // what its test needs; the attempt after it, decoded ahead when there is idle time
        const bool has_label = CACHED && (u32)tid < per;
        u32 lab = CG_NONE;
        u64 a_cur = 0;
        u32 sci = 0, scj = 0, cuh = 0, cul = 0;   // coded sites with the spare bits set
        double c_invr = 0, c_fld = 0, ei = 0, ej = 0;
        bool tracked = false;             // ei, ej hold the current local energies of my two sites
        bool ni = false, nj = false;      // occupations of my two sites
        Prop nxt = {0, 0, 0, 0, 0};
        bool nxt_valid = false;
        u32 hl = 0;                       // hops consumed in this launch
        auto take = [&](const Prop& q) {
            cuh = q.uh; cul = q.ul;
            sci = q.ci | geo.spare; scj = q.cj | geo.spare;
            c_invr = tb.inv(q.k); c_fld = tb.field(q.k);
            tracked = false;
        };
        // occupations of a pair as of hop hl: the bitmap (complete up to hop nlow, never ahead of me) and the
        // newer hops replayed in order
        auto read_n = [&](u32 ci, u32 cj, bool& oi, bool& oj) {
            const u32 vl = *(volatile u32*)&cm->nlow;         // read before the bits (volatile accesses of one thread stay in order)
            const u32 si = geo.site(ci), sj = geo.site(cj);
            bool a = BIT((volatile u32*)s_n, si) != 0u, c = BIT((volatile u32*)s_n, sj) != 0u;
            for (u32 h = vl + 1u; h <= hl; ++h) {
                const uint2 k = lds64u(&cm->hops[h % CG_HR][0]);
                if (ci == k.x) a = false; if (ci == k.y) a = true;
                if (cj == k.x) c = false; if (cj == k.y) c = true;
            }
            oi = a; oj = c;
        };
        // local energies of a pair as of hop hl: a snapshot that is complete on every CTA + the newer hops' terms
        auto read_eps = [&](u32 sc_i, u32 sc_j, double& oi, double& oj) {
            const u32 v = ld_acquire_cta(&cm->ver);
            u32 buf = cur0 + v % CG_RING; if (buf >= CG_RING) buf -= CG_RING;
            const double* __restrict__ erd = p.eps[buf];
            double a = ld_cg(erd + geo.site(sc_i & mask)), c = ld_cg(erd + geo.site(sc_j & mask));
            for (u32 h = (v << Hs) + 1u; h <= hl; ++h) {
                const uint2 k = lds64u(&cm->hops[h % CG_HR][0]);
                a = __dadd_rn(a, hop_term(tf, mask, sc_i, k.x, k.y));
                c = __dadd_rn(c, hop_term(tf, mask, sc_j, k.x, k.y));
            }
            oi = a; oj = c;
        };
        // MULTI: logical slot k (1 .. KX) holds attempt a_cur + k P, label lab + k P; it sits in physical slot
        // (rot + k - 1) mod KX, so that a consumed slot 0 is replaced by rotating (per thread)
        u32 rot = 0;
        bool mh = false; u32 mhi = 0, mhj = 0;    // the hop consumed last, not yet applied to slots 1 .. KX
        auto xidx = [&](u32 k) { u32 ph = rot + k - 1u; if (ph >= KX) ph -= KX; return ph * (u32)TW + (u32)tid; };
        auto x_decode = [&](u32 k) {              // as of hop hl
            const Prop q = decode_attempt(tb, p, geo, a_cur + (u64)k * P);
            const u32 ix = xidx(k);
            bool oi, oj;
            read_n(q.ci, q.cj, oi, oj);
            x_ci[ix] = q.ci | geo.spare; x_cj[ix] = q.cj | geo.spare; x_uh[ix] = q.uh; x_ul[ix] = q.ul; x_k[ix] = q.k;
            x_fl[ix] = 8u | (oi ? 1u : 0u) | (oj ? 2u : 0u);
        };
        if (has_label) {
            const u32 g = b * per + (u32)tid, g0 = c_first * per + t0r;
            lab = g >= g0 ? g - g0 : g + P - g0;
            a_cur = a_start + lab;
            take(decode_attempt(tb, p, geo, a_cur));
            read_n(sci & mask, scj & mask, ni, nj);
            if (MULTI) for (u32 k = 1; k <= KX; ++k) x_decode(k);
        }

        Slab<TW, RP> slab;
        {
            const u32 c0 = cur0;
            slab.load(p.eps[c0], p.work, pr0, pr1, geo, (u32)tid);
        }
        u64 a0 = a_start;                 // first attempt of the window (used when labels are not cached)
        bool upd = false, last = false;
        bool fresh = false;               // my attempt was consumed: the next one is not taken over yet
        bool inflight = false;            // the slab's gathers of hop hs are in flight
        u32 hz = 0, hw = 0, hs = 0;       // coded sites of the hop whose slab update is pending; hop the slab is working on
        double a_i = 0, b_i = 0, a_j = 0, b_j = 0;    // gathers in flight for the followed pair
        bool addterm = false;
        u64 t_test = 0, t_slab = 0, t_wait = 0;
        long long tprev = TIMED ? clock64() : 0;
        // take over the next attempt (decoded ahead of time as a rule) and the occupations of its pair
        auto refresh = [&]() {
            if (!nxt_valid) nxt = decode_attempt(tb, p, geo, a_cur);
            take(nxt); nxt_valid = false;
            read_n(sci & mask, scj & mask, ni, nj);
            fresh = false;
        };
        // the test of my proposal on the current state (steps 1-2)
        // A proposal starts to follow its two energies (one snapshot read + the pending hops' terms) while it is
        // still Mt - M labels away from the window, so that this never happens on the path of an iteration's result
        const u32 Mt = min(P, max(2u * M, M + 4096u));
        auto test_mine = [&](u32& best) {
            const bool th = lab < Mt && ni && !nj;                // theta_ij, inside the window or about to enter it
            if (th) {
                if (!tracked) { read_eps(sci, scj, ei, ej); tracked = true; }
                else if (addterm) {           // the term of the hop consumed last (gathered when it was consumed)
                    ei = __dadd_rn(ei, __dsub_rn(a_i, b_i)); ej = __dadd_rn(ej, __dsub_rn(a_j, b_j));
                }
                if (lab < M) {
                    // dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
                    const double dE = __dsub_rn(__dsub_rn(__dsub_rn(ej, ei), c_invr), c_fld);
                    if (metropolis(dE, cuh, cul, p.T, p.inv_T)) best = lab;
                }
            } else tracked = false;
        };
        for (u32 e = 0;; ++e) {
            const u32 xs = e % CG_XR, e32 = e_start + e;
            // ---- steps 1-2: propose and test on S_e, state untouched
            u32 best = CG_NONE, bi = 0, bj = 0;
            bool far_ = false;
            if (CACHED) {
                // A thread whose attempt was consumed takes over its next one when its warp is far from the front of the
                // window (below, behind the result); only if the new label lies inside the window already - P - used or more,
                // so hardly ever - it has to happen before the test
                if (fresh && lab < M) refresh();
                if (has_label && !fresh) test_mine(best);
                addterm = false;
                bi = sci & mask; bj = scj & mask;
                if (MULTI && has_label) {
                    // slots 1 .. KX: the hop consumed last (occupations, followed energies), then the test
                    const u32 si = mhi | geo.spare, sj = mhj | geo.spare;
                    // the four table gathers of a followed slot are issued one slot ahead of their use
                    // (the slots are visited in physical order: the lowest accepting label does not depend on the order)
                    u32 n_ix = (u32)tid, n_fl = x_fl[n_ix], n_ci = x_ci[n_ix], n_cj = x_cj[n_ix];
                    u32 k = KX + 1u - rot; if (k > KX) k -= KX;     // logical slot in physical slot 0
                    double g0 = 0, g1 = 0, g2 = 0, g3 = 0;
                    auto gather = [&]() {
                        if (mh && (n_fl & 12u) == 12u) {
                            g0 = __ldg(tf + ((n_ci - mhj) & mask)); g1 = __ldg(tf + ((n_ci - mhi) & mask));
                            g2 = __ldg(tf + ((n_cj - mhj) & mask)); g3 = __ldg(tf + ((n_cj - mhi) & mask));
                        }
                    };
                    gather();
                    for (u32 ph = 0; ph < KX; ++ph, k = (k == KX ? 1u : k + 1u)) {
                        const u32 labk = lab + k * P;
                        const u32 ix = n_ix;
                        u32 fl = n_fl;
                        const u32 ci_ = n_ci, cj_ = n_cj;
                        const double t0 = g0, t1 = g1, t2 = g2, t3 = g3;
                        if (ph + 1u < KX) { n_ix += (u32)TW; n_fl = x_fl[n_ix]; n_ci = x_ci[n_ix]; n_cj = x_cj[n_ix]; gather(); }
                        if (!(fl & 8u)) {
                            if (labk >= M) continue;            // decoded later, when the warp is far from the front
                            x_decode(k); fl = x_fl[ix];
                        } else if (mh) {
                            if (fl & 4u) {
                                x_ei[ix] = __dadd_rn(x_ei[ix], __dsub_rn(t0, t1));
                                x_ej[ix] = __dadd_rn(x_ej[ix], __dsub_rn(t2, t3));
                            }
                            if (ci_ == si) fl &= ~1u; if (ci_ == sj) fl |= 1u;
                            if (cj_ == si) fl &= ~2u; if (cj_ == sj) fl |= 2u;
                        }
                        if (labk < M && (fl & 3u) == 1u) {     // theta_ij, inside the window
                            const u32 ci_ = x_ci[ix], cj_ = x_cj[ix];     // (a slot decoded just now: not the values read ahead)
                            double vi, vj;
                            if (!(fl & 4u)) { read_eps(ci_, cj_, vi, vj); x_ei[ix] = vi; x_ej[ix] = vj; fl |= 4u; }
                            else { vi = x_ei[ix]; vj = x_ej[ix]; }
                            const u32 kk = x_k[ix];
                            const double dE = __dsub_rn(__dsub_rn(__dsub_rn(vj, vi), tb.inv(kk)), tb.field(kk));
                            if (labk < best && metropolis(dE, x_uh[ix], x_ul[ix], p.T, p.inv_T)) {
                                best = labk; bi = ci_ & mask; bj = cj_ & mask;
                            }
                        } else fl &= ~4u;
                        x_fl[ix] = fl;
                    }
                    mh = false;
                }
                far_ = __reduce_min_sync(CG_FULL, lab) >= min(CG_FRONT, P >> 2);               // warp-uniform
                u32 wmin = __reduce_min_sync(CG_FULL, best);
                // ---- step 3: lowest accepting label of the warp, for the collector
                if (wmin == CG_NONE ? lane == 0 : best == wmin) {   // labels are distinct: one lane
                    sts128(&cm->res[e % (2 * CG_XR)][warp][0], ((u64)e32 << 32) | wmin, ((u64)bi << 32) | (u64)bj);
                }
            } else {
                for (u32 l = lab0 + tid; l < lab1; l += TW) {
                    const Prop q = decode_attempt(tb, p, geo, a0 + l);
                    bool oi, oj;
                    read_n(q.ci, q.cj, oi, oj);
                    if (!oi || oj) continue;                                     // theta_ij
                    double vi, vj;
                    read_eps(q.ci | geo.spare, q.cj | geo.spare, vi, vj);
                    const double dE = __dsub_rn(__dsub_rn(__dsub_rn(vj, vi), tb.inv(q.k)), tb.field(q.k));
                    if (metropolis(dE, q.uh, q.ul, p.T, p.inv_T)) { best = l; bi = q.ci; bj = q.cj; break; }
                }
                const u32 wmin = __reduce_min_sync(CG_FULL, best);
                if (wmin == CG_NONE ? lane == 0 : best == wmin) {
                    sts128(&cm->res[e % (2 * CG_XR)][warp][0], ((u64)e32 << 32) | wmin, ((u64)bi << 32) | (u64)bj);
                }
            }
            long long t1 = 0;
            if (TIMED) { t1 = clock64(); t_test += (u64)(t1 - tprev); }
            // ---- step 3b for my part of the slab: the hop consumed last (its table gathers were
            // issued when it was consumed, behind those of the followed pair); first the decode one attempt ahead
            // (a warp near the front of the window is on the critical path of the next iterations: its decode waits
            // until all of its labels have been consumed and it sits at the far end of the window)
            if (CACHED && far_) {
                if (fresh) refresh();
                if (!MULTI && has_label && !nxt_valid) { nxt = decode_attempt(tb, p, geo, a_cur + P); nxt_valid = true; }
                if (MULTI && has_label)
                    for (u32 k = 1; k <= KX; ++k) if (!(x_fl[xidx(k)] & 8u)) x_decode(k);
            }
            // The slab runs one hop behind: the gathers of the hop consumed last are issued here, behind the result, and
            // were issued one iteration ago for the hop that is finished now - their latency is never waited for, and
            // nothing of the slab sits between the outcome and the test.
            if (inflight) {
                const bool snap = (hs & Hm) == 0u;
                u32 buf = cur0 + (hs >> Hs) % CG_RING; if (buf >= CG_RING) buf -= CG_RING;
                slab.finish(tf, mask, geo, p.work, snap ? p.eps[buf] : nullptr, pr0, pr1);
                if (snap) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&cm->pubbar[((hs >> Hs) - 1u) % CG_PB]);
                }
                inflight = false;
            }
            if (upd) { slab.issue(tf, mask, hz, hw); hs = hl; inflight = true; upd = false; }
            long long t2 = 0;
            if (TIMED) { t2 = clock64(); t_slab += (u64)(t2 - t1); }
            if (last) break;
            // ---- O_e
            if (!mbar_wait(&cm->full[xs], (e / CG_XR) & 1u, p, cm, 8u)) return;
            const uint4 d = lds128u(&cm->desc[xs]);        // used, flags, ci, cj
            __syncwarp();
            if (lane == 0) mbar_arrive(&cm->empty[xs]);
            if (TIMED) { tprev = clock64(); t_wait += (u64)(tprev - t2); }
            if (d.y & CG_F_ABORT) return;
            last = (d.y & CG_F_LAST) != 0u;
            if (MULTI && has_label) {
                // labels first: a consumed slot 0 is replaced by the lowest slot that survives (its state is that of
                // S_e, like slot 0's), to which the hop of O_e is then applied below like to any slot 0
                if (lab >= d.x) lab -= d.x;
                else {
                    const u32 c = (d.x - lab + P - 1u) / P;        // consumed slots: labels lab + k P < used, 1 <= c <= K
                    fresh = true; tracked = false; addterm = false;
                    if (c <= KX) {
                        const u32 ix = xidx(c);
                        const u32 fl = x_fl[ix];
                        if (fl & 8u) {
                            sci = x_ci[ix]; scj = x_cj[ix]; cuh = x_uh[ix]; cul = x_ul[ix];
                            const u32 kk = x_k[ix];
                            c_invr = tb.inv(kk); c_fld = tb.field(kk);
                            ni = (fl & 1u) != 0u; nj = (fl & 2u) != 0u; tracked = (fl & 4u) != 0u;
                            if (tracked) { ei = x_ei[ix]; ej = x_ej[ix]; }
                            fresh = false;
                        }
                    }
                    lab += c * P - d.x; a_cur += (u64)c * P;
                    rot += c; while (rot >= KX) rot -= KX;
                    for (u32 k = (c <= KX ? KX + 1u - c : 1u); k <= KX; ++k) x_fl[xidx(k)] = 0u;
                }
            }
            if (d.y & CG_F_HOP) {
                if (MULTI) { mh = true; mhi = d.z; mhj = d.w; }
                if (CACHED) {
                    // the term of this hop for the pair I follow: the four gathers come first (discarded if my
                    // attempt was consumed or theta_ij turns out to have changed), then the slab's
                    if (tracked) {
                        a_i = __ldg(tf + ((sci - d.w) & mask)); b_i = __ldg(tf + ((sci - d.z) & mask));
                        a_j = __ldg(tf + ((scj - d.w) & mask)); b_j = __ldg(tf + ((scj - d.z) & mask));
                        addterm = true;
                    }
                    const u32 si = d.z | geo.spare, sj = d.w | geo.spare;
                    if (sci == si) ni = false; if (sci == sj) ni = true;
                    if (scj == si) nj = false; if (scj == sj) nj = true;
                }
                ++hl; upd = true; hz = d.z; hw = d.w;
            }
            if (CACHED && !MULTI) {
                if (has_label) {
                    if (lab >= d.x) lab -= d.x;
                    else {                              // my attempt was consumed: the next one, P attempts later
                        lab += P - d.x; a_cur += P;
                        fresh = true; tracked = false; addterm = false;
                    }
                }
            } else if (!CACHED) a0 += d.x;
        }
        if (inflight) {                   // the last hop of the launch
            const bool snap = (hs & Hm) == 0u;
            u32 buf = cur0 + (hs >> Hs) % CG_RING; if (buf >= CG_RING) buf -= CG_RING;
            slab.finish(tf, mask, geo, p.work, snap ? p.eps[buf] : nullptr, pr0, pr1);
            if (snap) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&cm->pubbar[((hs >> Hs) - 1u) % CG_PB]);
            }
        }
        // the final state of my part of the slab, unless the last hop was a snapshot anyway
        if (n_hops & Hm) {
            u32 buf = cur0 + (n_snaps + 1u) % CG_RING; if (buf >= CG_RING) buf -= CG_RING;
            slab.flush(p.work, p.eps[buf], pr0, pr1);
        }
        if (TIMED && b == 0 && lane == 0) {
            atomicAdd(&p.ctl->cyc_propose, t_test); atomicAdd(&p.ctl->cyc_update, t_slab);
            atomicAdd(&p.ctl->cyc_wait, t_wait); atomicAdd(&p.ctl->cyc_warps, 1ull);
        }
    }
    // every warp but the exchange warp: the two barriers of the end of the launch (skipped when it was abandoned:
    // the exchange warp is then not there)
    if (*(volatile u32*)&cm->abort) return;
    asm volatile("bar.sync 1, %0;" ::"r"(THREADS) : "memory");
    asm volatile("bar.sync 2, %0;" ::"r"(THREADS) : "memory");
    if (csz > 1) cluster_sync_all();
}

template <int NW, int RP, bool CACHED, bool TIMED, bool MULTI = false>
__global__ void __launch_bounds__(NW * 32 + 96, 1) cg_pr_persistent(const CgParams p)
{
    pr_persistent_body<NW, RP, CACHED, TIMED, MULTI>(p, blockIdx.x, gridDim.x);
}

// Replica packing (the paper recommends averaging many samples): ONE launch,
// CTAs [first[s], first[s+1]) run sim s with its own parameter block.  The sims share nothing.
template <int NW, int RP, bool CACHED>
__global__ void __launch_bounds__(NW * 32 + 96, 1)
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
    pr_persistent_body<NW, RP, CACHED, false>(sp, s_b, s_nb);
}

// ---- a sim that fits ONE CTA: everything in shared memory, two CTA barriers per iteration ------------------------
// Small lattices (the paper recommends averaging many samples) have no exchange between CTAs to hide, so
// the dataflow between role warps above only costs them hand-overs.  Here all CG_ST threads are workers.  Thread t owns
// the attempts a = t (mod CG_ST) and keeps its proposal decoded; eps and the occupation bitmap live in shared memory,
// so a test (steps 1-2) reads eps_i, eps_j and n_i, n_j afresh (no followed energies, no pending
// terms), the lowest accepting label (step 3) is ONE 64-bit shared-memory atomicMin of (label, thread), and after the
// barrier every thread adds the hop's term to its sites of eps (step 3b: the same single rounded add per
// site and hop as everywhere else).  Second barrier, next iteration.
#define CG_ST 512           // threads (= labels held) of the single-CTA kernel; 1024 for 512 < M <= 1024
#define CG_SINGLE_MAX_N 8192u   // eps in shared memory: 64 KiB
template <int ST>
__device__ __forceinline__ void pr_single_body(const CgParams& p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int KS = p.Ksm;
    u64* s_cdfi = reinterpret_cast<u64*>(smem_raw);
    double* s_invr = reinterpret_cast<double*>(s_cdfi + KS);
    double* s_fld = s_invr + KS;
    double* s_eps = s_fld + KS;
    u32* s_disp = reinterpret_cast<u32*>(s_eps + p.N);
    u32* s_guide = s_disp + KS;
    u32* s_n = s_guide + CG_GUIDE;
    __shared__ u32 s_key[3];               // lowest accepting label of iterations e, e+1, e+2 (mod 3); thread = (label + g0) mod ST
    __shared__ __align__(8) u32 s_sites[2][ST][2];   // coded sites of every thread's proposal, by iteration parity
    const Tables tb = {s_cdfi, s_invr, s_fld, s_disp, s_guide, p.cdfi, p.invr_k, p.fld_k, p.disp, (u32)KS};
    const Geo geo = {p.hi1, p.hi2, p.spare, p.mask, (u32)(p.L - 1), p.lgL};
    const int tid = threadIdx.x, lane = tid & 31;
    const u32 N = p.N, M = p.M, mask = p.mask, P = ST;
    const double* __restrict__ tf = p.tf;
    CgCtl* const ctl = p.ctl;
    double* const g_eps = p.eps[ctl->cur];

    for (int k = tid; k < KS; k += ST) {
        s_cdfi[k] = p.cdfi[k]; s_invr[k] = p.invr_k[k]; s_fld[k] = p.fld_k[k]; s_disp[k] = p.disp[k];
    }
    for (int k = tid; k < CG_GUIDE; k += ST) s_guide[k] = p.guide[k];
    for (u32 w = tid; w < (N + 31) / 32; w += ST) s_n[w] = p.nbits[w];
    for (u32 k = tid; k < N; k += ST) s_eps[k] = __ldcg(g_eps + k);
    if (tid < 3) s_key[tid] = CG_NONE;
    const u64 a_start = ctl->attempts, hops_start = ctl->hops, log_base = ctl->log_base;
    const u32 n_hops = p.n_hops;
    __syncthreads();

    // my attempt and the one after it (a proposal is a pure function of seed and attempt index)
    u32 g0 = (u32)(a_start % P);          // the thread that holds the first label of the window
    u32 lab = ((u32)tid - g0) & (P - 1u);
    u64 a_cur = a_start + lab;
    // the attempt after mine is decoded in two halves while my label lies outside the window (nothing to test then):
    // stage 0 = nothing yet, 1 = random words drawn, 2 = complete
    Prop cur = decode_attempt(tb, p, geo, a_cur), nxt = decode_attempt(tb, p, geo, a_cur + P);
    u32 stage = 2; u64 nxt_m = 0;
    double c_invr = tb.inv(cur.k), c_fld = tb.field(cur.k);
    u32 c_si = geo.site(cur.ci), c_sj = geo.site(cur.cj);
    u32 hc = 0, e = 0, k3 = 0;             // e: iterations mod 2^32 (parity of the site buffers only), k3 = iterations mod 3
    u64 its = 0;
    u64 used_sum = 0;
    long long dP = 0;
    while (hc < n_hops) {
        // ---- steps 1-2: test my proposal on the current state
        sts64u(&s_sites[e & 1u][tid][0], cur.ci, cur.cj);
        u32 best = CG_NONE;
        if (lab < M) {
            if (BIT(s_n, c_si) && !BIT(s_n, c_sj)) {                      // theta_ij
                // dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
                const double dE = __dsub_rn(__dsub_rn(__dsub_rn(s_eps[c_sj], s_eps[c_si]), c_invr), c_fld);
                if (metropolis(dE, cur.uh, cur.ul, p.T, p.inv_T)) best = lab;
            }
        }
        // a warp with nothing to test draws half of its lanes' next decode per iteration (in a warp that tests, the decode would
        // lengthen the path to the barrier: measured 1159 k against 1340 k hops/s at config 1)
        if (__all_sync(CG_FULL, lab >= M)) {
            if (stage == 0u) { nxt = decode_words(p, geo, a_cur + P, nxt_m); stage = 1u; }
            else if (stage == 1u) { decode_finish(tb, geo, nxt, nxt_m); stage = 2u; }
        }
        // ---- step 3: the lowest accepting label; labels are distinct
        const u32 wmin = __reduce_min_sync(CG_FULL, best);
        const u32 k3n = k3 == 2u ? 0u : k3 + 1u;
        if (wmin != CG_NONE && lane == 0) atomicMin(&s_key[k3], wmin);
        if (tid == 0) s_key[k3n] = CG_NONE;                                // last read before the previous barrier pair
        __syncthreads();
        const u32 key = s_key[k3];
        k3 = k3n;
        const bool hop = key != CG_NONE;
        const u32 used = hop ? key + 1u : M;                               // m = (p-1) M + q
        if (hop) {
            const uint2 w = lds64u(&s_sites[e & 1u][(key + g0) & (P - 1u)][0]);      // coded sites of the executed hop
            // step 3b: eps_l += 1/r_lj - 1/r_li, difference first, then ONE add
            for (u32 l = tid; l < N; l += ST)
                s_eps[l] = __dadd_rn(s_eps[l], hop_term(tf, mask, geo.code(l) | geo.spare, w.x, w.y));
            ++hc;
            if (tid == ST - 1) {                                        // step 3a, dP, hop log (a thread with few sites)
                const u32 hi_ = geo.site(w.x), hj_ = geo.site(w.y);
                s_n[hi_ >> 5] &= ~(1u << (hi_ & 31));
                s_n[hj_ >> 5] |= 1u << (hj_ & 31);
                dP += geo.dx(hi_, hj_);
                const u64 h = hops_start + hc - 1u - log_base;
                if (h < p.log_cap) { p.log_a[h] = a_start + used_sum + used - 1; p.log_i[h] = hi_; p.log_j[h] = hj_; }
            }
        }
        used_sum += used;
        g0 = (g0 + used) & (P - 1u);
        ++e; ++its;
        if (lab >= used) lab -= used;
        else {                                                             // consumed: my next attempt, P attempts later
            if (stage == 0u) nxt = decode_words(p, geo, a_cur + P, nxt_m);       // (M close to P: no idle iterations)
            if (stage != 2u) decode_finish(tb, geo, nxt, nxt_m);
            lab += P - used; a_cur += P;
            cur = nxt; c_invr = tb.inv(cur.k); c_fld = tb.field(cur.k);
            c_si = geo.site(cur.ci); c_sj = geo.site(cur.cj);
            stage = 0u;
        }
        __syncthreads();
    }
    for (u32 k = tid; k < N; k += ST) __stcg(g_eps + k, s_eps[k]);
    for (u32 w = tid; w < (N + 31) / 32; w += ST) p.nbits[w] = s_n[w];
    if (tid == ST - 1) {
        ctl->attempts = a_start + used_sum; ctl->hops = hops_start + hc;
        ctl->iterations += its; ctl->proposals += (u64)M * its;
        ctl->dP += dP; ctl->epoch += its;
    }
}

template <int ST>
__global__ void __launch_bounds__(ST, 1) cg_pr_single(const CgParams p) { pr_single_body<ST>(p); }

// many single-CTA sims in one launch: CTA s runs sim s
template <int ST>
__global__ void __launch_bounds__(ST, 1) cg_pr_single_many(const CgParams* __restrict__ ps)
{
    __shared__ CgParams sp;
    if (threadIdx.x == 0) sp = ps[blockIdx.x];
    __syncthreads();
    pr_single_body<ST>(sp);
}

// ---- the single-CTA kernel with KL labels per thread: lattices up to N = 16384 on ONE SM (replica packing) --------
// Same idea as cg_pr_single (eps, occupations and tower in shared memory, two CTA barriers per iteration), for
// M <= KL x 512 labels: thread t holds the attempts a, a + 512, .., a + (KL-1) 512 (labels lab + j 512) in registers
// and tests all of them in every iteration.  The lowest accepting label and its two coded sites travel in ONE 64-bit
// shared-memory atomicMin (label << 42 | c_i << 21 | c_j).  A consumed slot 0 is replaced by shifting the slots down and
// decoding a new top one.  Slower per sim than the dataflow kernel on 8-32 SMs, but it takes one SM: 148 lattices of
// L = 128 run side by side (cg_run_many).
#define CG_SK_MAX_N 16384u
template <int KL>
__device__ __forceinline__ void pr_singlek_body(const CgParams& p)
{
    constexpr int ST = CG_ST;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int KS = p.Ksm;
    u64* s_cdfi = reinterpret_cast<u64*>(smem_raw);
    double* s_invr = reinterpret_cast<double*>(s_cdfi + KS);
    double* s_fld = s_invr + KS;
    double* s_eps = s_fld + KS;
    u32* s_disp = reinterpret_cast<u32*>(s_eps + p.N);
    u32* s_guide = s_disp + KS;
    u32* s_n = s_guide + CG_GUIDE;
    __shared__ u64 s_key[3];
    const Tables tb = {s_cdfi, s_invr, s_fld, s_disp, s_guide, p.cdfi, p.invr_k, p.fld_k, p.disp, (u32)KS};
    const Geo geo = {p.hi1, p.hi2, p.spare, p.mask, (u32)(p.L - 1), p.lgL};
    const int tid = threadIdx.x, lane = tid & 31;
    const u32 N = p.N, M = p.M, mask = p.mask, P = ST;
    const double* __restrict__ tf = p.tf;
    CgCtl* const ctl = p.ctl;
    double* const g_eps = p.eps[ctl->cur];

    for (int k = tid; k < KS; k += ST) {
        s_cdfi[k] = p.cdfi[k]; s_invr[k] = p.invr_k[k]; s_fld[k] = p.fld_k[k]; s_disp[k] = p.disp[k];
    }
    for (int k = tid; k < CG_GUIDE; k += ST) s_guide[k] = p.guide[k];
    for (u32 w = tid; w < (N + 31) / 32; w += ST) s_n[w] = p.nbits[w];
    for (u32 k = tid; k < N; k += ST) s_eps[k] = __ldcg(g_eps + k);
    if (tid < 3) s_key[tid] = ~0ull;
    const u64 a_start = ctl->attempts, hops_start = ctl->hops, log_base = ctl->log_base;
    const u32 n_hops = p.n_hops;
    __syncthreads();

    const u32 g0 = (u32)(a_start % P);
    u32 lab = ((u32)tid - g0) & (P - 1u);          // label of slot 0; slot j holds label lab + j P
    u64 a_cur = a_start + lab;
    u32 cci[KL], ccj[KL], cuh[KL], cul[KL], ck[KL];
#pragma unroll
    for (int j = 0; j < KL; ++j) {
        const Prop q = decode_attempt(tb, p, geo, a_cur + (u64)j * P);
        cci[j] = q.ci; ccj[j] = q.cj; cuh[j] = q.uh; cul[j] = q.ul; ck[j] = q.k;
    }
    u32 hc = 0, k3 = 0;
    u64 its = 0, used_sum = 0;
    long long dP = 0;
    while (hc < n_hops) {
        // ---- steps 1-2 for my KL labels, step 3: lowest accepting label
        u64 best = ~0ull;
#pragma unroll
        for (int j = 0; j < KL; ++j) {
            const u32 labj = lab + (u32)j * P;
            if (labj < M) {
                const u32 si = geo.site(cci[j]), sj = geo.site(ccj[j]);
                if (BIT(s_n, si) && !BIT(s_n, sj)) {
                    const double dE = __dsub_rn(__dsub_rn(__dsub_rn(s_eps[sj], s_eps[si]), tb.inv(ck[j])), tb.field(ck[j]));
                    if (metropolis(dE, cuh[j], cul[j], p.T, p.inv_T))
                        best = min(best, ((u64)labj << 42) | ((u64)cci[j] << 21) | (u64)ccj[j]);
                }
            }
        }
        const u32 blab = (u32)(best >> 42);            // 0x3FFFFF when nothing accepted
        const u32 wmin = __reduce_min_sync(CG_FULL, blab);
        const u32 k3n = k3 == 2u ? 0u : k3 + 1u;
        if (best != ~0ull && blab == wmin) atomicMin(&s_key[k3], best);
        if (tid == 0) s_key[k3n] = ~0ull;
        __syncthreads();
        const u64 key = s_key[k3];
        k3 = k3n;
        const bool hop = key != ~0ull;
        const u32 used = hop ? (u32)(key >> 42) + 1u : M;
        if (hop) {
            const u32 wci = (u32)(key >> 21) & 0x1FFFFFu, wcj = (u32)key & 0x1FFFFFu;
            // step 3b: eps_l += 1/r_lj - 1/r_li, difference first, then ONE add.  (The folded table in shared
            // memory instead of the unfolded one through L1/L2 was measured slower, 22.1 M against 24.2 M hops/s for 148 sims of
            // L = 128: the update is bound by its instruction count, 16384 sites on one SM, not by the table traffic.)
            for (u32 l = tid; l < N; l += ST)
                s_eps[l] = __dadd_rn(s_eps[l], hop_term(tf, mask, geo.code(l) | geo.spare, wci, wcj));
            ++hc;
            if (tid == ST - 1) {
                const u32 hi_ = geo.site(wci), hj_ = geo.site(wcj);
                s_n[hi_ >> 5] &= ~(1u << (hi_ & 31));
                s_n[hj_ >> 5] |= 1u << (hj_ & 31);
                dP += geo.dx(hi_, hj_);
                const u64 h = hops_start + hc - 1u - log_base;
                if (h < p.log_cap) { p.log_a[h] = a_start + used_sum + used - 1; p.log_i[h] = hi_; p.log_j[h] = hj_; }
            }
        }
        used_sum += used;
        ++its;
        if (lab >= used) lab -= used;
        else {
            // slots whose labels are consumed: lab + j P < used, j < c; the others move down, new ones are decoded at the top
            const u32 c = (used - lab + P - 1u) / P;      // 1 <= c <= KL
            for (u32 r = 0; r < c; ++r) {
#pragma unroll
                for (int j = 0; j + 1 < KL; ++j) { cci[j] = cci[j + 1]; ccj[j] = ccj[j + 1]; cuh[j] = cuh[j + 1]; cul[j] = cul[j + 1]; ck[j] = ck[j + 1]; }
                const Prop q = decode_attempt(tb, p, geo, a_cur + (u64)(KL + r) * P);
                cci[KL - 1] = q.ci; ccj[KL - 1] = q.cj; cuh[KL - 1] = q.uh; cul[KL - 1] = q.ul; ck[KL - 1] = q.k;
            }
            lab += c * P - used; a_cur += (u64)c * P;
        }
        __syncthreads();
    }
    for (u32 k = tid; k < N; k += ST) __stcg(g_eps + k, s_eps[k]);
    for (u32 w = tid; w < (N + 31) / 32; w += ST) p.nbits[w] = s_n[w];
    if (tid == ST - 1) {
        ctl->attempts = a_start + used_sum; ctl->hops = hops_start + hc;
        ctl->iterations += its; ctl->proposals += (u64)M * its;
        ctl->dP += dP; ctl->epoch += its;
    }
}

template <int KL>
__global__ void __launch_bounds__(CG_ST, 1) cg_pr_singlek(const CgParams p) { pr_singlek_body<KL>(p); }
template <int KL>
__global__ void __launch_bounds__(CG_ST, 1) cg_pr_singlek_many(const CgParams* __restrict__ ps)
{
    __shared__ CgParams sp;
    if (threadIdx.x == 0) sp = ps[blockIdx.x];
    __syncthreads();
    pr_singlek_body<KL>(sp);
}

__device__ __forceinline__ Geo make_geo(const CgParams& p)
{
    const Geo g = {p.hi1, p.hi2, p.spare, p.mask, (u32)(p.L - 1), p.lgL};
    return g;
}

// Step a6 alone: scripted hops, update in place (no readers), one launch.
template <int THREADS, int RP>
__global__ void __launch_bounds__(THREADS, 1)
cg_update_scripted(const CgParams p, const u32* __restrict__ hop_i, const u32* __restrict__ hop_j, u64 count)
{
    const u32 b = blockIdx.x, nb = gridDim.x;
    const Geo geo = make_geo(p);
    const u32 pairs = p.N / 2, pper = (pairs + nb - 1) / nb;
    const u32 pr0 = min(pairs, b * pper), pr1 = min(pairs, pr0 + pper);
    double* e = p.eps[p.ctl->cur];
    Slab<THREADS, RP> slab;
    slab.load(e, e, pr0, pr1, geo, threadIdx.x);
    for (u64 h = 0; h < count; ++h) {
        slab.issue(p.tf, p.mask, geo.code(__ldg(hop_i + h)), geo.code(__ldg(hop_j + h)));
        slab.finish(p.tf, p.mask, geo, e, e, pr0, pr1);
    }
    if (b == 0 && threadIdx.x == 0) {       // occupations and dipole moment, in hop order
        long long dP = p.ctl->dP; u32 bad = 0;
        for (u64 h = 0; h < count; ++h) {
            const u32 i = hop_i[h], j = hop_j[h];
            const u32 wi = p.nbits[i >> 5], wj = p.nbits[j >> 5];
            if (!((wi >> (i & 31)) & 1u) || ((wj >> (j & 31)) & 1u)) ++bad;
            p.nbits[i >> 5] &= ~(1u << (i & 31));
            p.nbits[j >> 5] |= (1u << (j & 31));
            dP += geo.dx(i, j);
        }
        p.ctl->dP = dP; p.ctl->hops += count; p.ctl->bad_hops += bad;
    }
}


// Step a6 alone, staged (include/cg.h: cg_apply_hops).  CTA b owns `rows` whole lattice rows (z, y) and keeps their eps in
// shared memory.  For an executed hop i -> j the sites of lattice row (z, y) need the table row of the offset
// ((z - z_j) mod L, (y - y_j) mod L) - L contiguous doubles, 16-byte aligned - read at (x - x_j) mod L, and the same for i:
// two bulk copies per lattice row (cp.async.bulk, completion counted on an mbarrier) bring them into one of NST stages in
// shared memory, issued NST - 1 hops ahead by the first warp; every warp then forms eps += 1/r_lj - 1/r_li from shared
// memory only: no thread waits for a global load, and the load/store units see no gathers at all.  Every table entry of a
// hop is fetched exactly once by the whole grid (16 N bytes of table traffic per hop, through the copy engine).
template <int THREADS, int NST>
__global__ void __launch_bounds__(THREADS)
cg_update_staged(const CgParams p, const u32* __restrict__ hop_i, const u32* __restrict__ hop_j, u64 count, u32 rows)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) u64 full[NST], empty[NST];
    const Geo geo = make_geo(p);
    const u32 L = (u32)p.L, lg = (u32)p.lgL, Lm = L - 1u, mask = p.mask;
    const u32 total_rows = p.N >> lg;
    const u32 row0 = blockIdx.x * rows, n_rows = min(rows, total_rows - min(total_rows, row0));
    const u32 s_lo = row0 << lg, n_s = n_rows << lg;
    double* const sl = reinterpret_cast<double*>(smem_raw);                  // the slab: rows x L
    double* const stage = sl + (size_t)rows * L;                             // [NST][2 ends][rows][L]
    const u32 st_sz = 2u * rows * L;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* e = p.eps[p.ctl->cur];
    if (threadIdx.x == 0)
        for (int k = 0; k < NST; ++k) { mbar_init(&full[k], 1); mbar_init(&empty[k], THREADS / 32); }
    for (u32 k = threadIdx.x; k < n_s; k += THREADS) sl[k] = __ldcg(e + s_lo + k);
    __syncthreads();
    const double* __restrict__ tf = p.tf;
    // the table rows of hop h into stage h % NST (first warp)
    auto fetch = [&](u64 h) {
        const u32 st = (u32)(h % NST), use = (u32)(h / NST);
        if (use >= 1u) mbar_spin(&empty[st], (use - 1u) & 1u);
        if (lane == 0) mbar_expect_tx(&full[st], 2u * n_rows * 8u * L);
        __syncwarp();
        const u32 ci = geo.code(__ldg(hop_i + h)), cj = geo.code(__ldg(hop_j + h));
        const u32 cjr = cj & ~Lm, cir = ci & ~Lm;                            // hop sites with x = 0
        double* const dj = stage + st * st_sz;
        double* const di = dj + rows * L;
        for (u32 r = (u32)lane; r < 2u * n_rows; r += 32u) {
            const u32 rr = r >> 1, isj = r & 1u;
            const u32 rc = geo.code((row0 + rr) << lg) | geo.spare;          // first site of the lattice row
            bulk_g2s((isj ? dj : di) + rr * L, tf + ((rc - (isj ? cjr : cir)) & mask), 8u * L, &full[st]);
        }
    };
    if (n_rows) {
        if (warp == 0) for (u64 h = 0; h < (u64)(NST - 1) && h < count; ++h) fetch(h);
        for (u64 h = 0; h < count; ++h) {
            if (warp == 0 && h + NST - 1 < count) fetch(h + NST - 1);
            const u32 st = (u32)(h % NST);
            mbar_spin(&full[st], (u32)(h / NST) & 1u);
            const double* __restrict__ sj = stage + st * st_sz;
            const double* __restrict__ si = sj + rows * L;
            const u32 xi = __ldg(hop_i + h) & Lm, xj = __ldg(hop_j + h) & Lm;
#pragma unroll 4
            for (u32 k = threadIdx.x; k < n_s; k += THREADS) {
                const u32 r = k & ~Lm;                                       // row offset; x = k & Lm
                sl[k] = __dadd_rn(sl[k], __dsub_rn(sj[r + ((k - xj) & Lm)], si[r + ((k - xi) & Lm)]));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
        }
        for (u32 k = threadIdx.x; k < n_s; k += THREADS) __stcg(e + s_lo + k, sl[k]);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {       // occupations and dipole moment, in hop order
        long long dP = p.ctl->dP; u32 bad = 0;
        for (u64 h = 0; h < count; ++h) {
            const u32 i = hop_i[h], j = hop_j[h];
            const u32 wi = p.nbits[i >> 5], wj = p.nbits[j >> 5];
            if (!((wi >> (i & 31)) & 1u) || ((wj >> (j & 31)) & 1u)) ++bad;
            p.nbits[i >> 5] &= ~(1u << (i & 31));
            p.nbits[j >> 5] |= (1u << (j & 31));
            dP += geo.dx(i, j);
        }
        p.ctl->dP = dP; p.ctl->hops += count; p.ctl->bad_hops += bad;
    }
}

// ---- one-time set-up (step a0) --------------------------------------------------------------

// tf from the folded table: entry (dz, dy, dx) of the unfolded index space (fields of width 2L)
__global__ void cg_build_tf(const double* __restrict__ tq, double* __restrict__ tf, int L, int lg, int Lz, int pitch, u32 total)
{
    for (u32 idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const int dx = idx & (2 * L - 1), dy = (idx >> (lg + 1)) & (2 * L - 1), dz = idx >> (2 * lg + 2);
        double v = 0.0;
        if (dx < L && dy < L && dz < Lz) {
            const int fx = min(dx, L - dx), fy = min(dy, L - dy), fz = min(dz, Lz - dz);
            v = tq[((size_t)fz * pitch + fy) * pitch + fx];
        }
        tf[idx] = v;
    }
}

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
                                int L, int lg, int Lz, int pitch, u32 N)
{
    const u32 s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    const int z = s >> (2 * lg), y = (s >> lg) & (L - 1), x = s & (L - 1);
    double e = phi[s];
    u32 word = 0;
    for (int zt = 0; zt < Lz; ++zt) {
        int dz = (z - zt) & (Lz - 1); dz = min(dz, Lz - dz);
        for (int yt = 0; yt < L; ++yt) {
            int dy = (y - yt) & (L - 1); dy = min(dy, L - dy);
            const double* row = tq + ((size_t)dz * pitch + dy) * pitch;
            for (int xt = 0; xt < L; ++xt) {
                const u32 t = ((((u32)zt << lg) | (u32)yt) << lg) | (u32)xt;
                if ((t & 31u) == 0u || xt == 0) word = __ldg(nbits + (t >> 5));
                int dx = (x - xt) & (L - 1); dx = min(dx, L - dx);
                const double half = __dmul_rn(0.5, __ldg(row + dx));  // exact; 0 on the diagonal
                e = ((word >> (t & 31u)) & 1u) ? __dadd_rn(e, half) : __dsub_rn(e, half);
            }
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

// L2 roofline probes: L1-bypassing accesses over a resident buffer, `reps` passes inside one launch.
// mode 0: read-modify-write, 1: read only (the sum is kept alive through `sink`), 2: write only;
// VEC = 16 or 32 bytes per access.
template <int VEC>
__global__ void cg_l2_probe(double* buf, size_t nvec, int reps, int mode, double* sink)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (int r = 0; r < reps; ++r)
        for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nvec; k += stride) {
            if (VEC == 16) {
                double2* q = reinterpret_cast<double2*>(buf) + k;
                double2 v = make_double2((double)r, 1.0);
                if (mode != 2) v = __ldcg(q);
                if (mode == 1) acc += v.x + v.y;
                else { v.x += 1.0; v.y -= 1.0; __stcg(q, v); }
            } else {
                double* q = buf + 4 * k;
                double a = (double)r, b = 1.0, c = 2.0, d = 3.0;
                if (mode != 2)
                    asm volatile("ld.global.cg.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(q) : "memory");
                if (mode == 1) acc += (a + b) + (c + d);
                else {
                    a += 1.0; b -= 1.0; c += 1.0; d -= 1.0;
                    asm volatile("st.global.cg.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(q), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
                }
            }
        }
    if (mode == 1 && acc == 123.456) *sink = acc;
}

// -------------------------------------------------------------------- host --

struct cg_sim {
    int dim = 2, L = 0, Lz = 1, lgL = 0, pitch = 0;
    u32 N = 0, M = 0;
    double W = 0, xi = 0, T = 0, E = 0;
    u64 seed = 0;
    // host tables (live part of the tower)
    int64_t K = 0, Klive = 0;
    std::vector<int32_t> dz, dy, dx;
    std::vector<double> cdf, invr_k, fld_k;
    std::vector<u64> cdfi;
    std::vector<u32> guide;
    double S = 0, Gamma = 0;
    u32 hi1 = 0, hi2 = 0, spare = 0, mask = 0, tf_len = 0;
    // device
    int device = 0;
    cudaStream_t stream = nullptr;
    void* ws = nullptr; bool own_ws = false;
    double* d_eps[CG_RING] = {};
    double* d_work = nullptr; double* d_scratch = nullptr; double* d_phi = nullptr;
    u32* d_nbits = nullptr; double* d_tq = nullptr; double* d_tf = nullptr;
    u64* d_cdfi = nullptr; double* d_invr_k = nullptr; double* d_fld_k = nullptr; u32* d_disp = nullptr;
    u32* d_guide = nullptr;
    u64* d_slots = nullptr; CgCtl* d_ctl = nullptr; u64* d_red = nullptr;
    void* d_log = nullptr; bool own_log = false; u64 log_cap = 0;
    bool log_gap = false;                 // scripted hops (cg_apply_hops) were executed while the log was on: it no longer holds every hop
    void* d_many = nullptr; size_t many_cap = 0;      // parameter blocks of cg_run_many (owned by its first sim)
    // launch shape and tuning
    int num_sms = 0, n_ctas = 0, threads = 0, smem = 0, rp = 0, pl = 0;   // pl > 0: cached proposals
    int lpt = 1;                          // cached labels per thread (> 1: the MULTI kernel, M > n_ctas * pl)
    bool single = false;                  // the single-CTA kernel (cg_pr_single): 1 CTA x CG_ST threads, state in shared memory
    int snap_shift = 3;                   // snapshots every 1 << snap_shift hops
    bool snap_auto = true;                // not set by cg_set_tuning: chosen from the lattice size at init
    int cluster = 1;                      // CTAs per thread-block cluster in use
    int cluster_pref = 0;                 // cg_set_tuning: 0 = automatic (clusters when the whole sim fits a few of them)
    bool timers = false;                  // cg_set_phase_timers
    int update_kernel = 0;                // cg_set_update_kernel: 0 automatic, 1 gathers, 2 staged
    int smem_optin = 0;
    u64 watchdog_ns = 10ull * 1000 * 1000 * 1000;
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

// supported lattices: L a power of two, 2D 4..1024, 3D 4..64 (N <= 2^20: the occupation bitmap of the whole
// lattice lives in every CTA's shared memory)
static bool valid_L(int dim, int L, int* lg)
{
    if (L < 4 || L > (dim == 3 ? 64 : 1024) || (L & (L - 1))) return false;
    int k = 0; while ((1 << k) < L) ++k;
    if (lg) *lg = k;
    return true;
}

struct WsLayout { size_t eps0, work, scratch, phi, nbits, tq, tf, cdfi, invr_k, fld_k, disp, guide, slots, ctl, red, total; };
#define CG_SLOT_BYTES ((size_t)8 * CG_SLOT_U64 * CG_MAX_CTAS)

static WsLayout ws_layout(int dim, int L)
{
    const size_t N = dim == 3 ? (size_t)L * L * L : (size_t)L * L;
    const size_t h = (size_t)L / 2 + 1, hz = dim == 3 ? h : 1;
    const size_t tf_len = dim == 3 ? 4 * N : 2 * N;     // index space of the unfolded table (fields of width 2L)
    const size_t kcap = std::min<size_t>(N, 65536);     // the live tower is capped at 65535 entries
    WsLayout w; size_t o = 0;
    w.eps0 = o; o += CG_RING * align256(8 * N);
    w.work = o; o += align256(8 * N);
    w.scratch = o; o += align256(8 * N);
    w.phi = o; o += align256(8 * N);
    w.nbits = o; o += align256(N / 8 + 4);
    w.tq = o; o += align256(8 * hz * h * h);
    w.tf = o; o += align256(8 * tf_len);
    w.cdfi = o; o += align256(8 * kcap);
    w.invr_k = o; o += align256(8 * kcap);
    w.fld_k = o; o += align256(8 * kcap);
    w.disp = o; o += align256(4 * kcap);
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
    if (!valid_L(2, L, nullptr)) return 0;
    return ws_layout(2, L).total;
}

extern "C" size_t cg_workspace_bytes3(int L, uint32_t M)
{
    (void)M;
    if (!valid_L(3, L, nullptr)) return 0;
    return ws_layout(3, L).total;
}

static u32 host_code(const cg_sim* s, u32 site) { return site + (site & s->hi1) + ((site & s->hi2) << 1); }

// Displacement list, tower and Gamma on the host.
static void build_tables(cg_sim* s, std::vector<double>& tq)
{
    const int L = s->L, h = L / 2, Lz = s->Lz;
    struct D { long long r2; int dz, dy, dx; };
    std::vector<D> d;
    const int zlo = Lz == 1 ? 0 : -h + 1, zhi = Lz == 1 ? 0 : h;
    for (int dz = zlo; dz <= zhi; ++dz)
        for (int dy = -h + 1; dy <= h; ++dy)
            for (int dx = -h + 1; dx <= h; ++dx) {
                const long long r2 = (long long)dz * dz + (long long)dy * dy + (long long)dx * dx;
                if (r2 > 0 && r2 <= (long long)h * h) d.push_back({r2, dz, dy, dx});
            }
    std::sort(d.begin(), d.end(), [](const D& a, const D& b) {
        if (a.r2 != b.r2) return a.r2 < b.r2;
        if (a.dz != b.dz) return a.dz < b.dz;
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
    s->dz.resize(live); s->dy.resize(live); s->dx.resize(live); s->cdf.resize(live); s->invr_k.resize(live);
    s->fld_k.resize(live); s->cdfi.resize(live);
    for (size_t k = 0; k < live; ++k) {
        s->dz[k] = d[k].dz; s->dy[k] = d[k].dy; s->dx[k] = d[k].dx;
        s->cdf[k] = (k + 1 == K) ? 1.0 : run[k] / acc;
        s->invr_k[k] = 1.0 / std::sqrt((double)d[k].r2);
        s->fld_k[k] = s->E * (double)d[k].dx;              // the field term of dH
    }
    s->cdf[live - 1] = 1.0;
    // u_d = m 2^-43 with integer m < 2^43, so u_d < cdf_k <=> m < ceil(cdf_k 2^43) (scaling by a power
    // of two and ceil are exact in double)
    for (size_t k = 0; k < live; ++k) s->cdfi[k] = (u64)std::ceil(std::ldexp(s->cdf[k], 43));
    // Guide over t = 2^43 - m: bucket = (binade of t, next 3 bits).  The tail of the tower is geometric
    // in r, so every bucket brackets only a few k; both ends found by bisection.
    auto kstar = [&](u64 m) {
        return (u32)(std::upper_bound(s->cdfi.begin(), s->cdfi.end(), m) - s->cdfi.begin());   // smallest k with m < cdfi_k
    };
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
    const int pitch = s->pitch, hz = Lz == 1 ? 1 : pitch;
    tq.assign((size_t)hz * pitch * pitch, 0.0);
    for (int c = 0; c < hz; ++c)
        for (int a = 0; a <= h; ++a)
            for (int b = 0; b <= h; ++b) {
                const long long r2 = (long long)c * c + (long long)a * a + (long long)b * b;
                tq[((size_t)c * pitch + a) * pitch + b] = r2 ? 1.0 / std::sqrt((double)r2) : 0.0;
            }
}

static size_t smem_base_bytes(const cg_sim* s)
{
    const size_t ks = (size_t)std::min<int64_t>(s->Klive, CG_KS);
    return ks * 28 + 4 * CG_GUIDE + 4 * (((size_t)s->N + 31) / 32) + 16;
}
// K labels per thread: K - 1 extra slots of CG_XSLOT_BYTES for each of the 448 worker threads, 16-byte aligned
static size_t smem_xoff(const cg_sim* s) { return (smem_base_bytes(s) + 15) & ~(size_t)15; }
static size_t smem_bytes(const cg_sim* s, int K)
{
    return K > 1 ? smem_xoff(s) + (size_t)(K - 1) * 448 * CG_XSLOT_BYTES : smem_base_bytes(s);
}

// hops between snapshots -> gate distance G with CG_RING H > 2 G + 2 H - 2 (pr_persistent_body, "Snapshots")
static u32 gate_for(int snap_shift)
{
    static const u32 g[4] = {5, 8, 8, 16};
    return g[snap_shift];
}
static_assert(CG_RING * 1 > 2 * 5 + 2 * 1 - 2 && CG_RING * 2 > 2 * 8 + 2 * 2 - 2 && CG_RING * 4 > 2 * 8 + 2 * 4 - 2
              && CG_RING * 8 > 2 * 16 + 2 * 8 - 2, "snapshot ring too short for the gate");
static_assert(CG_HR > CG_XR + 16 + CG_MAX_SNAP - 1, "hop ring too short");
static_assert(CG_SRING > 16 + CG_MAX_SNAP + CG_XR, "slot ring too short");
static_assert(CG_PB > 16 / CG_MAX_SNAP + 1 && CG_PB > 5 + 1, "publication barriers");

static CgParams make_params(const cg_sim* s, u32 n_hops)
{
    CgParams p;
    for (int k = 0; k < CG_RING; ++k) p.eps[k] = s->d_eps[k];
    p.work = s->d_work;
    p.tf = s->d_tf; p.tq = s->d_tq; p.nbits = s->d_nbits;
    p.cdfi = s->d_cdfi; p.invr_k = s->d_invr_k; p.fld_k = s->d_fld_k; p.disp = s->d_disp;
    p.guide = s->d_guide;
    p.slots = s->d_slots; p.ctl = s->d_ctl;
    p.log_a = (u64*)s->d_log;
    p.log_i = s->d_log ? (u32*)((char*)s->d_log + 8 * s->log_cap) : nullptr;
    p.log_j = s->d_log ? (u32*)((char*)s->d_log + 12 * s->log_cap) : nullptr;
    p.log_cap = s->d_log ? s->log_cap : 0;
    p.L = s->L; p.lgL = s->lgL; p.Klive = (int)s->Klive; p.Ksm = (int)std::min<int64_t>(s->Klive, CG_KS);
    p.hi1 = s->hi1; p.hi2 = s->hi2; p.spare = s->spare; p.mask = s->mask;
    p.N = s->N; p.M = s->M; p.PL = (u32)s->pl;
    p.seed_lo = (u32)s->seed; p.seed_hi = (u32)(s->seed >> 32);
    p.T = s->T; p.E = s->E; p.inv_T = (float)(1.0 / s->T); p.n_hops = n_hops;
    p.snap_shift = (u32)s->snap_shift; p.gate = gate_for(s->snap_shift);
    p.cluster = (u32)s->cluster; p.watchdog_ns = s->watchdog_ns;
    p.K = (u32)s->lpt; p.xoff = (u32)smem_xoff(s);
    return p;
}

typedef void (*persist_fn)(const CgParams);
typedef void (*scripted_fn)(const CgParams, const u32*, const u32*, u64);

// RP = eps pairs a thread keeps in registers (0: the slab lives in a working buffer in global memory);
// TIMED: with the phase timers of cg_get_phase_cycles (544-thread shapes only)
template <int NW, bool CACHED, bool TIMED>
static persist_fn persistent_kernel_t(int rp)
{
    switch (rp) {
        case 0: return cg_pr_persistent<NW, 0, CACHED, TIMED>;
        case 1: return cg_pr_persistent<NW, 1, CACHED, TIMED>;
        case 2: return cg_pr_persistent<NW, 2, CACHED, TIMED>;
        case 4: if (NW <= 16) return cg_pr_persistent<NW <= 16 ? NW : 5, 4, CACHED, NW <= 16 ? TIMED : false>; break;
        case 8: if (NW <= 14) return cg_pr_persistent<NW <= 14 ? NW : 5, 8, CACHED, NW <= 14 ? TIMED : false>; break;
    }
    return nullptr;
}
// threads per CTA = 32 (worker warps + 3): 256 (5), 544 (14), 608 (16), 1024 (29)
static int workers_of(int threads)
{
    switch (threads) { case 256: return 5; case 544: return 14; case 608: return 16; case 1024: return 29; }
    return 0;
}
static persist_fn persistent_kernel(int threads, int rp, bool cached, bool timed, bool multi = false)
{
    if (multi) {                          // several cached labels per thread: 544-thread shape only, no phase timers
        if (threads != 544 || !cached) return nullptr;
        switch (rp) {
            case 0: return cg_pr_persistent<14, 0, true, false, true>;
            case 1: return cg_pr_persistent<14, 1, true, false, true>;
            case 2: return cg_pr_persistent<14, 2, true, false, true>;
            case 4: return cg_pr_persistent<14, 4, true, false, true>;
            case 8: return cg_pr_persistent<14, 8, true, false, true>;
        }
        return nullptr;
    }
    switch (workers_of(threads)) {
        case 5: return cached ? persistent_kernel_t<5, true, false>(rp) : persistent_kernel_t<5, false, false>(rp);
        case 14: if (timed) return cached ? persistent_kernel_t<14, true, true>(rp) : persistent_kernel_t<14, false, true>(rp);
                 return cached ? persistent_kernel_t<14, true, false>(rp) : persistent_kernel_t<14, false, false>(rp);
        case 16: return cached ? persistent_kernel_t<16, true, false>(rp) : persistent_kernel_t<16, false, false>(rp);
        case 29: return cached ? persistent_kernel_t<29, true, false>(rp) : persistent_kernel_t<29, false, false>(rp);
    }
    return nullptr;
}
typedef void (*many_fn)(const CgParams*, const u32*, u32);
template <bool CACHED>
static many_fn many_kernel_t(int rp)
{
    switch (rp) {
        case 0: return cg_pr_persistent_many<14, 0, CACHED>;
        case 1: return cg_pr_persistent_many<14, 1, CACHED>;
        case 2: return cg_pr_persistent_many<14, 2, CACHED>;
        case 4: return cg_pr_persistent_many<14, 4, CACHED>;
        case 8: return cg_pr_persistent_many<14, 8, CACHED>;
    }
    return nullptr;
}
static many_fn many_kernel(int threads, int rp, bool cached)
{
    if (threads != 544) return nullptr;
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

// smallest supported register tiling that holds `pairs` pairs per CTA on `workers` threads, else 0
static int choose_rp(u64 pairs, int n_ctas, int workers, int cap)
{
    const u64 per_cta = (pairs + n_ctas - 1) / n_ctas;
    const u64 need = (per_cta + workers - 1) / workers;
    for (int rp = 1; rp <= cap; rp *= 2)
        if ((u64)rp >= need) return rp;
    return 0;
}
static int rp_cap(int threads) { return threads == 1024 ? 2 : threads == 608 ? 4 : 8; }

// how many CTAs of this shape can be co-resident (in clusters of s->cluster)
static int max_coresident(cg_sim* s, int threads, int rp, bool cached, int K, int* out)
{
    const int smem = (int)smem_bytes(s, K);
    persist_fn f = persistent_kernel(threads, rp, cached, false, K > 1);
    if (!f) return CG_EINVAL;
    CK(cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    persist_fn ft = threads == 544 && K == 1 ? persistent_kernel(threads, rp, cached, true) : nullptr;      // the timed build
    if (ft) CK(cudaFuncSetAttribute((const void*)ft, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (s->cluster > 1) {
        if (s->cluster > 8) {
            CK(cudaFuncSetAttribute((const void*)f, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
            if (ft) CK(cudaFuncSetAttribute((const void*)ft, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        }
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(s->cluster * s->num_sms); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = (size_t)smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)s->cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nc = 0;
        CK(cudaOccupancyMaxActiveClusters(&nc, (const void*)f, &cfg));
        *out = std::min(nc * s->cluster, CG_MAX_CTAS);
        return CG_OK;
    }
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)f, threads, smem));
    *out = std::min(per_sm * s->num_sms, CG_MAX_CTAS);
    return CG_OK;
}

static int choose_launch_cs(cg_sim* s, int n_ctas, int threads)
{
    const bool auto_threads = threads == 0;
    if (auto_threads) threads = 544;
    if (!workers_of(threads)) return CG_EINVAL;
    const bool heuristic = n_ctas == 0;
    const int cs = s->cluster;
    for (int attempt = 0; attempt < 2; ++attempt) {
        const int workers = 32 * workers_of(threads);
        int want = n_ctas;
        if (heuristic) {
            const u64 work = std::max<u64>(s->M, s->N / 2);        // labels or pairs of sites, per worker thread
            want = (int)std::min<u64>((work + workers - 1) / workers, (u64)s->num_sms);
            want = std::max(1, want);
            want = (want + cs - 1) / cs * cs;
        }
        if (want < 1 || want > CG_MAX_CTAS || want % cs) return CG_EINVAL;
        int rp = choose_rp(s->N / 2, want, workers, rp_cap(threads));
        // labels cached in the threads: one each when M <= P = CTAs x workers, up to CG_KMAX each (MULTI kernel, 544-thread
        // shape) while they fit shared memory; beyond that every label is recomputed in every iteration
        auto labels_per_thread = [&](int ctas) {
            const u64 Pn = (u64)ctas * (u64)workers;
            if (s->M <= Pn) return 1;
            const u64 K = (s->M + Pn - 1) / Pn;
            if (threads != 544 || K > CG_KMAX) return 0;
            if (smem_bytes(s, (int)K) + sizeof(Comm) + 1024 > (size_t)s->smem_optin) return 0;
            return (int)K;
        };
        int K = labels_per_thread(want);
        bool cached = K >= 1;
        int cap = 0;
        int rc = max_coresident(s, threads, rp, cached, std::max(K, 1), &cap);
        if (rc != CG_OK) return rc;
        if (cap < cs) { s->err = "persistent kernel does not fit on the device in this cluster size"; return CG_EUNSUPPORTED; }
        if (want > cap) {
            if (!heuristic) return CG_EINVAL;
            want = cap / cs * cs;
            rp = choose_rp(s->N / 2, want, workers, rp_cap(threads));
            K = labels_per_thread(want);
            cached = K >= 1;
            rc = max_coresident(s, threads, rp, cached, std::max(K, 1), &cap);
            if (rc != CG_OK) return rc;
            if (want > cap) return CG_EUNSUPPORTED;
        }
        // clusters strand SMs: if the labels no longer fit the threads, larger CTAs keep them cached
        if (heuristic && auto_threads && K != 1 && threads == 544 && s->M <= (u64)want * 512u) { threads = 608; continue; }
        if (want != s->n_ctas)    // slots of CTAs that no longer exist must not look published
            CK(cudaMemsetAsync(s->d_slots, 0, CG_SLOT_BYTES, s->stream));
        s->n_ctas = want; s->threads = threads; s->rp = rp; s->pl = cached ? workers : 0;
        s->lpt = std::max(K, 1); s->smem = (int)smem_bytes(s, s->lpt);
        return CG_OK;
    }
    return CG_EUNSUPPORTED;
}

// Launch shape for (n_ctas, threads), 0 = heuristic, with the cluster size of cg_set_tuning.  Automatic cluster size
// (measured): CTAs of one cluster post through shared memory instead of L2, worth 6-8 % when the whole sim
// sits in one or a few clusters; on B200 clusters of 8 and 16 leave 28 and 36 of the 148 SMs unused, so a sim that
// wants every SM runs in pairs (+2 % at config 5, +15 % at config 4 with M = 65536).  An explicit CTA count keeps the largest cluster size that divides it.
// shared memory of the single-CTA kernel: tower head, guide, bitmap and eps
static size_t smem_single_bytes(const cg_sim* s) { return smem_base_bytes(s) + 8 * (size_t)s->N + 16; }

static int choose_launch(cg_sim* s, int n_ctas, int threads)
{
    // A sim whose labels and sites fit one CTA runs in the single-CTA kernel (everything in shared memory): chosen
    // automatically, or asked for as (1 CTA, CG_ST threads); any other explicit shape keeps the dataflow kernel.
    {
        // CG_ST threads hold up to CG_ST labels; 2 CG_ST threads (registers: 64 each) hold up to 2 CG_ST
        const int st = s->M <= CG_ST ? CG_ST : 2 * CG_ST;
        const bool fits = s->M <= 2 * CG_ST && s->N <= CG_SINGLE_MAX_N
                          && smem_single_bytes(s) + 12 * 1024 <= (size_t)s->smem_optin;
        // asked for: (1 CTA, 512 threads), or (1 CTA, 1024 threads) when 512 < M <= 1024 fits (else that is a dataflow shape);
        // automatic: up to 1024 sites (measured: at L = 64 the dataflow kernel on 8 CTAs is the faster one for a single sim,
        // 662 k against 508 k hops/s at M = 1024, but the single-CTA kernel takes one SM instead of eight: replica packing)
        const bool asked = threads == CG_ST && n_ctas <= 1;
        const bool asked2 = threads == 2 * CG_ST && n_ctas == 1 && fits && st == 2 * CG_ST;
        const bool automatic = threads == 0 && n_ctas == 0 && s->cluster_pref == 0 && s->N <= 2 * CG_ST && s->M <= 2 * CG_ST;
        if (asked && (st != CG_ST || s->N > CG_SINGLE_MAX_N)) {
            // more than 512 labels on 512 threads: the variant with 2, 4 or 8 labels per thread (lattices up to N = 16384 on one SM)
            const int kl = s->M <= 2 * CG_ST ? 2 : s->M <= 4 * CG_ST ? 4 : 8;
            const int smem = (int)(smem_base_bytes(s) + 8 * (size_t)s->N + 16);
            if (s->M > 8 * CG_ST || s->N > CG_SK_MAX_N || (size_t)smem + 4 * 1024 > (size_t)s->smem_optin) return CG_EINVAL;
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek_many<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek_many<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_singlek_many<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            s->single = true; s->n_ctas = 1; s->threads = CG_ST; s->rp = 0; s->pl = CG_ST; s->lpt = kl; s->smem = smem;
            s->cluster = 1;
            return CG_OK;
        }
        if (asked && !fits) return CG_EINVAL;
        if (fits && (asked || asked2 || automatic)) {
            const int smem = (int)smem_single_bytes(s);
            CK(cudaFuncSetAttribute((const void*)cg_pr_single<CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_single_many<CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_single<2 * CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            CK(cudaFuncSetAttribute((const void*)cg_pr_single_many<2 * CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            s->single = true; s->n_ctas = 1; s->threads = st; s->rp = 0; s->pl = st; s->lpt = 1; s->smem = smem;
            s->cluster = 1;
            return CG_OK;
        }
        s->single = false;
    }
    const int old = s->cluster;
    int cs = s->cluster_pref;
    if (cs == 0) {
        s->cluster = 1;
        int rc = choose_launch_cs(s, n_ctas, threads);
        if (rc != CG_OK) { s->cluster = old; return rc; }
        if (s->n_ctas < 2) return CG_OK;
        if (s->n_ctas > 96) cs = 2;       // pairs pack the 148 SMs exactly: half of the changes of decider stay inside a cluster
        else {
            cs = 16;
            if (n_ctas == 0) while (cs > 1 && cs / 2 >= s->n_ctas) cs /= 2;     // 5 CTAs -> one cluster of 8
        }
    }
    if (n_ctas) while (cs > 1 && n_ctas % cs) cs /= 2;
    for (; cs >= 1; cs /= 2) {
        s->cluster = cs;
        const int rc = choose_launch_cs(s, n_ctas, threads);
        if (rc == CG_OK) return CG_OK;
        if (s->cluster_pref != 0 || cs == 1) { s->cluster = old; return rc; }
    }
    s->cluster = old;
    return CG_EUNSUPPORTED;
}

static int init_impl(cg_sim** out, int dim, int L, double W, double xi, double T, double E, uint64_t seed,
                     uint32_t M, void* dev_ws, size_t bytes, void* stream, bool own)
{
    if (!out) return CG_EINVAL;
    *out = nullptr;
    if (L < 2 || (L & 1)) return CG_EINVAL;
    if (!(xi > 0.0) || !(T > 0.0) || !(W >= 0.0) || M < 1 || !std::isfinite(E) || !std::isfinite(W)
        || !std::isfinite(xi) || !std::isfinite(T)) return CG_EINVAL;
    int lg = 0;
    if (!valid_L(dim, L, &lg)) return CG_EUNSUPPORTED;
    if (M > (1u << 27)) return CG_EUNSUPPORTED;            // labels travel in 32-bit records next to other fields
    cg_sim* s = new (std::nothrow) cg_sim();
    if (!s) return CG_ENOMEM;
    struct Guard { cg_sim* s; ~Guard() { if (s) cg_free(s); } } guard{s};
    s->dim = dim; s->L = L; s->Lz = dim == 3 ? L : 1; s->lgL = lg; s->pitch = L / 2 + 1;
    s->N = dim == 3 ? (u32)L * (u32)L * (u32)L : (u32)L * (u32)L; s->M = M;
    s->W = W; s->xi = xi; s->T = T; s->E = E; s->seed = seed;
    s->stream = (cudaStream_t)stream;
    // site coding: c(s) = (z 2L + y) 2L + x (csrc: struct Geo)
    s->hi1 = ~(u32)(L - 1);
    s->hi2 = dim == 3 ? ~(u32)(L * L - 1) : 0u;
    s->spare = (u32)L | (dim == 3 ? (u32)(2 * L * L) : 0u);
    s->mask = (u32)(L - 1) | ((u32)(L - 1) << (lg + 1)) | (dim == 3 ? (u32)(L - 1) << (2 * lg + 2) : 0u);
    s->tf_len = dim == 3 ? 4u * s->N : 2u * s->N;
    if (const char* w = getenv("CG_WATCHDOG_MS")) s->watchdog_ns = (u64)strtoull(w, nullptr, 10) * 1000000ull;

    cudaDeviceProp prop;
    CK(cudaGetDevice(&s->device));
    CK(cudaGetDeviceProperties(&prop, s->device));
    s->num_sms = prop.multiProcessorCount;
    s->smem_optin = (int)prop.sharedMemPerBlockOptin;
    if (!prop.cooperativeLaunch) { s->err = "device lacks cooperative launch"; return CG_EUNSUPPORTED; }

    std::vector<double> tq;
    try { build_tables(s, tq); } catch (const std::bad_alloc&) { return CG_ENOMEM; }
    if (s->Klive > 65535) return CG_EUNSUPPORTED;           // the guide packs k in 16 bits
    s->smem = (int)smem_bytes(s, 1);
    if ((size_t)s->smem + sizeof(Comm) + 1024 > (size_t)prop.sharedMemPerBlockOptin) return CG_EUNSUPPORTED;

    const WsLayout w = ws_layout(dim, L);
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
    s->d_work = (double*)(base + w.work);
    s->d_scratch = (double*)(base + w.scratch); s->d_phi = (double*)(base + w.phi);
    s->d_nbits = (u32*)(base + w.nbits); s->d_tq = (double*)(base + w.tq); s->d_tf = (double*)(base + w.tf);
    s->d_cdfi = (u64*)(base + w.cdfi); s->d_invr_k = (double*)(base + w.invr_k);
    s->d_fld_k = (double*)(base + w.fld_k); s->d_guide = (u32*)(base + w.guide);
    s->d_disp = (u32*)(base + w.disp); s->d_slots = (u64*)(base + w.slots);
    s->d_ctl = (CgCtl*)(base + w.ctl); s->d_red = (u64*)(base + w.red);

    std::vector<u32> disp((size_t)s->Klive);
    for (int64_t k = 0; k < s->Klive; ++k) {
        const u32 mz = (u32)(s->dz[k] & (s->Lz - 1)), my = (u32)(s->dy[k] & (L - 1)), mx = (u32)(s->dx[k] & (L - 1));
        disp[k] = host_code(s, (((mz << lg) | my) << lg) | mx);
    }
    cudaStream_t st = s->stream;
    CK(cudaMemcpyAsync(s->d_tq, tq.data(), 8 * tq.size(), cudaMemcpyHostToDevice, st));
    cg_build_tf<<<std::min<u32>((s->tf_len + 255) / 256, 4096u), 256, 0, st>>>(s->d_tq, s->d_tf, L, lg, s->Lz, s->pitch, s->tf_len);
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
    const int ob = (int)std::min<u32>(N, 1024);          // N = 2^k >= 16, so ob divides N and is a warp multiple
    cg_init_occupations<<<N / ob, ob, 0, st>>>(keys, s->d_nbits, N);
    cg_full_sum_eps<<<(N + 127) / 128, 128, 0, st>>>(s->d_phi, s->d_nbits, s->d_tq, s->d_eps[0], L, lg, s->Lz, s->pitch, N);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));                        // host vectors above go out of scope

    // snapshot interval (measured): the 2 MiB of eps at N = 2^18 are worth writing through only every
    // 8 hops; smaller lattices run best with short pending lists
    s->snap_shift = s->N >= (1u << 18) ? 3 : 1;
    int rc = choose_launch(s, 0, 0);
    if (rc != CG_OK) return rc;
    guard.s = nullptr;
    *out = s;
    return CG_OK;
}

extern "C" int cg_init(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed, uint32_t M)
{
    return init_impl(out, 2, L, W, xi, T, E, seed, M, nullptr, 0, nullptr, true);
}

extern "C" int cg_init_ws(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed,
                          uint32_t M, void* dev_workspace, size_t bytes, void* cuda_stream)
{
    return init_impl(out, 2, L, W, xi, T, E, seed, M, dev_workspace, bytes, cuda_stream, false);
}

extern "C" int cg_init3(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed, uint32_t M)
{
    return init_impl(out, 3, L, W, xi, T, E, seed, M, nullptr, 0, nullptr, true);
}

extern "C" int cg_init3_ws(cg_sim** out, int L, double W, double xi, double T, double E, uint64_t seed,
                           uint32_t M, void* dev_workspace, size_t bytes, void* cuda_stream)
{
    return init_impl(out, 3, L, W, xi, T, E, seed, M, dev_workspace, bytes, cuda_stream, false);
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

// one cooperative launch, in clusters when the sim asks for them
static cudaError_t launch_coop(const void* f, int grid, int threads, int smem, cudaStream_t st, int cluster, void** args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = (size_t)smem; cfg.stream = st;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (cluster > 1) {
        at[1].id = cudaLaunchAttributeClusterDimension;
        at[1].val.clusterDim.x = (unsigned)cluster; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelExC(&cfg, f, args);
}

#ifndef CG_UPD_STAGES
#define CG_UPD_STAGES 6      // hops whose table rows are in flight in the staged update kernel
#endif
#ifndef CG_UPD_THREADS
#define CG_UPD_THREADS 128
#endif
#define CG_MAX_LAUNCH_HOPS (1u << 30)     // the kernel counts hops and iterations of one launch in 32 bits

extern "C" int cg_run(cg_sim* s, uint64_t n_hops)
{
    if (!s) return CG_EINVAL;
    if (s->single) {
        while (n_hops) {
            const u32 chunk = (u32)std::min<uint64_t>(n_hops, CG_MAX_LAUNCH_HOPS);
            const CgParams p = make_params(s, chunk);
            if (s->lpt == 2) cg_pr_singlek<2><<<1, CG_ST, (size_t)s->smem, s->stream>>>(p);
            else if (s->lpt == 4) cg_pr_singlek<4><<<1, CG_ST, (size_t)s->smem, s->stream>>>(p);
            else if (s->lpt == 8) cg_pr_singlek<8><<<1, CG_ST, (size_t)s->smem, s->stream>>>(p);
            else if (s->threads == CG_ST) cg_pr_single<CG_ST><<<1, CG_ST, (size_t)s->smem, s->stream>>>(p);
            else cg_pr_single<2 * CG_ST><<<1, 2 * CG_ST, (size_t)s->smem, s->stream>>>(p);
            CK(cudaGetLastError());
            n_hops -= chunk;
        }
        return CG_OK;
    }
    persist_fn f = persistent_kernel(s->threads, s->rp, s->pl > 0, s->timers && s->threads == 544 && s->lpt == 1, s->lpt > 1);
    if (!f) return CG_EINVAL;
    while (n_hops) {
        const u32 chunk = (u32)std::min<uint64_t>(n_hops, CG_MAX_LAUNCH_HOPS);
        CgParams p = make_params(s, chunk);
        void* args[] = {&p};
        CK(launch_coop((const void*)f, s->n_ctas, s->threads, s->smem, s->stream, s->cluster, args));
        n_hops -= chunk;
    }
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
        if (s->device != s0->device || s->stream != s0->stream || s->threads != s0->threads || s->rp != s0->rp
            || (s->pl > 0 && s->lpt == 1) != (s0->pl > 0 && s0->lpt == 1) || s->single != s0->single || (s->single && s->lpt != s0->lpt)) {
            s0->err = "cg_run_many: the sims must share device, stream and launch shape (threads, register tiling, "
                      "cached labels)";
            return CG_EINVAL;
        }
        first[(size_t)k + 1] = first[(size_t)k] + (u32)s->n_ctas;
        smem = std::max(smem, s->smem);
    }
    const bool single = s0->single;       // threads == CG_ST everywhere: single-CTA sims, which need not be co-resident
    many_fn f = single ? nullptr : many_kernel(s0->threads, s0->rp, s0->pl > 0 && s0->lpt == 1);     // several labels per thread: recomputed here
    if (!single && !f) { s0->err = "cg_run_many: only 544-thread launch shapes"; return CG_EUNSUPPORTED; }
    const u32 total = first[(size_t)n_sims];
    if (single) {
        CK0(s0, cudaFuncSetAttribute((const void*)cg_pr_single_many<CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK0(s0, cudaFuncSetAttribute((const void*)cg_pr_single_many<2 * CG_ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK0(s0, cudaFuncSetAttribute((const void*)cg_pr_singlek_many<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK0(s0, cudaFuncSetAttribute((const void*)cg_pr_singlek_many<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        CK0(s0, cudaFuncSetAttribute((const void*)cg_pr_singlek_many<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    } else {
        CK0(s0, cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        int per_sm = 0;
        CK0(s0, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)f, s0->threads, smem));
        if (total > (u32)(per_sm * s0->num_sms)) {     // every CTA of every sim must be resident: they wait for each other
            s0->err = "cg_run_many: the sims' CTAs do not fit on the device together";
            return CG_EUNSUPPORTED;
        }
    }
    const size_t need = ps.size() * sizeof(CgParams) + first.size() * sizeof(u32);
    if (s0->many_cap < need) {
        if (s0->d_many) { CK0(s0, cudaStreamSynchronize(s0->stream)); cudaFree(s0->d_many); s0->d_many = nullptr; s0->many_cap = 0; }
        CK0(s0, cudaMalloc(&s0->d_many, need));
        s0->many_cap = need;
    }
    CgParams* d_ps = (CgParams*)s0->d_many;
    u32* d_first = (u32*)((char*)s0->d_many + ps.size() * sizeof(CgParams));
    while (n_hops) {
        const u32 chunk = (u32)std::min<uint64_t>(n_hops, CG_MAX_LAUNCH_HOPS);
        for (int k = 0; k < n_sims; ++k) {
            ps[(size_t)k] = make_params(sims[k], chunk); ps[(size_t)k].cluster = 1;       // posts through L2
            if (sims[k]->lpt > 1) { ps[(size_t)k].PL = 0; ps[(size_t)k].K = 1; }
        }
        // pageable sources: the copies are staged before the calls return
        CK0(s0, cudaMemcpyAsync(d_ps, ps.data(), ps.size() * sizeof(CgParams), cudaMemcpyHostToDevice, s0->stream));
        CK0(s0, cudaMemcpyAsync(d_first, first.data(), first.size() * sizeof(u32), cudaMemcpyHostToDevice, s0->stream));
        u32 n = (u32)n_sims;
        void* args[] = {&d_ps, &d_first, &n};
        if (single) {
            if (s0->lpt == 2) cg_pr_singlek_many<2><<<(unsigned)n_sims, CG_ST, (size_t)smem, s0->stream>>>(d_ps);
            else if (s0->lpt == 4) cg_pr_singlek_many<4><<<(unsigned)n_sims, CG_ST, (size_t)smem, s0->stream>>>(d_ps);
            else if (s0->lpt == 8) cg_pr_singlek_many<8><<<(unsigned)n_sims, CG_ST, (size_t)smem, s0->stream>>>(d_ps);
            else if (s0->threads == CG_ST) cg_pr_single_many<CG_ST><<<(unsigned)n_sims, CG_ST, (size_t)smem, s0->stream>>>(d_ps);
            else cg_pr_single_many<2 * CG_ST><<<(unsigned)n_sims, 2 * CG_ST, (size_t)smem, s0->stream>>>(d_ps);
            CK0(s0, cudaGetLastError());
        } else
        CK0(s0, launch_coop((const void*)f, (int)total, s0->threads, smem, s0->stream, 1, args));
        n_hops -= chunk;
    }
    return CG_OK;
}

// the control block, after everything queued on the stream; CG_EDEVICE when a launch was abandoned
static int read_ctl(cg_sim* s, CgCtl* c)
{
    CK(cudaMemcpyAsync(c, s->d_ctl, sizeof *c, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (c->abort) {
        char buf[160];
        snprintf(buf, sizeof buf, "the persistent kernel gave up waiting (watchdog, wait %u); the state is undefined until "
                                  "cg_set_state", c->abort);
        s->err = buf;
        return CG_EDEVICE;
    }
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
    if (rc != CG_OK && rc != CG_EDEVICE) return rc;          // a new state is the way out of an abandoned launch
    c.attempts = attempts; c.hops = hops; c.dP = dP; c.iterations = 0; c.proposals = 0; c.cur = 0; c.abort = 0;
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
            if (bytes / 16 < capacity || ((uintptr_t)dev_buf & 7)) return CG_EINVAL;
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
    if (s->log_gap) return CG_EINVAL;                        // scripted hops are not logged: the indices would lie
    const u64 have = std::min<u64>(c.hops - c.log_base, s->log_cap);
    if (first > have || count > have - first) return CG_EINVAL;
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
                                                               s->L, s->lgL, s->Lz, s->pitch, s->N);
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

struct EventPair {          // released on every return path
    cudaEvent_t a = nullptr, b = nullptr;
    ~EventPair() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
};

extern "C" int cg_apply_hops(cg_sim* s, uint64_t count, const uint32_t* i, const uint32_t* j, float* ms)
{
    if (!s || (count && (!i || !j))) return CG_EINVAL;
    if (ms) *ms = 0.f;
    if (!count) return CG_OK;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    // theta_ij of every scripted hop, in hop order, BEFORE anything is touched
    {
        std::vector<u32> bits((s->N + 31) / 32);
        CK(cudaMemcpyAsync(bits.data(), s->d_nbits, 4 * bits.size(), cudaMemcpyDeviceToHost, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        for (u64 h = 0; h < count; ++h) {
            const u32 a = i[h], b = j[h];
            if (a >= s->N || b >= s->N || a == b) return CG_EINVAL;
            if (!((bits[a >> 5] >> (a & 31)) & 1u) || ((bits[b >> 5] >> (b & 31)) & 1u)) return CG_EINVAL;
            bits[a >> 5] &= ~(1u << (a & 31)); bits[b >> 5] |= 1u << (b & 31);
        }
    }
    u32* d_ij = nullptr;
    if (s->d_log) s->log_gap = true;
    CK(cudaMalloc(&d_ij, 8 * count));
    struct Free { void* p; ~Free() { cudaFree(p); } } fr{d_ij};
    CK(cudaMemcpyAsync(d_ij, i, 4 * count, cudaMemcpyHostToDevice, s->stream));
    CK(cudaMemcpyAsync(d_ij + count, j, 4 * count, cudaMemcpyHostToDevice, s->stream));
    EventPair ev;
    CK(cudaEventCreate(&ev.a)); CK(cudaEventCreate(&ev.b));
    CgParams p = make_params(s, 0);
    // many small CTAs per SM (one block of 64 sites per warp; 128 threads measured best) keep enough
    // requests in flight to make the stand-alone update throughput-bound; larger lattices fall back to
    // one CTA per SM
    const u64 g1 = (s->N / 2 + 127) / 128;
    const int grid = (int)std::max<u64>(1, std::min<u64>((s->N / 2 + 511) / 512, (u64)s->num_sms));
    // staged kernel: whole lattice rows per CTA, slab + CG_UPD_STAGES stages of two table rows per lattice row in shared memory
    // (many small CTAs - about 512 sites each, several per SM - keep more table rows in flight per SM than a few large ones)
    const u32 total_rows = s->N / (u32)s->L;
    const u32 rows = std::max(1u, 512u / (u32)s->L);
    const size_t st_smem = (size_t)rows * s->L * 8 * (1 + 2 * CG_UPD_STAGES);
    // measured on B200: the bulk copies of the rows saturate near 4 TB/s, the gather kernel is twice as fast (DESIGN.md
    // 6.2): the staged kernel runs only when asked for
    const bool fits = s->L >= 32 && st_smem + 1024 <= (size_t)s->smem_optin;
    if (s->update_kernel == 2 && !fits) return CG_EUNSUPPORTED;
    const bool staged = s->update_kernel == 2;
    if (staged) CK(cudaFuncSetAttribute((const void*)cg_update_staged<CG_UPD_THREADS, CG_UPD_STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)st_smem));
    CK(cudaEventRecord(ev.a, s->stream));
    if (staged) cg_update_staged<CG_UPD_THREADS, CG_UPD_STAGES><<<(total_rows + rows - 1) / rows, CG_UPD_THREADS, st_smem, s->stream>>>(p, d_ij, d_ij + count, count, rows);
    else if (g1 <= (u64)s->num_sms * 12) cg_update_scripted<128, 1><<<(int)g1, 128, 0, s->stream>>>(p, d_ij, d_ij + count, count);
    else scripted_kernel(choose_rp(s->N / 2, grid, 512, 8))<<<grid, 512, 0, s->stream>>>(p, d_ij, d_ij + count, count);
    CK(cudaEventRecord(ev.b, s->stream));
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(s->stream));
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, ev.a, ev.b));
    if (ms) *ms = t;
    rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (c.bad_hops) {                          // cannot happen after the check above; kept as a device-side assertion
        c.bad_hops = 0;
        CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        return CG_EINVAL;
    }
    return CG_OK;
}

extern "C" int cg_set_update_kernel(cg_sim* s, int kind)
{
    if (!s || kind < 0 || kind > 2) return CG_EINVAL;
    s->update_kernel = kind;
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

extern "C" int cg_get_table_dz(cg_sim* s, int32_t* dz)
{
    if (!s || !dz) return CG_EINVAL;
    memcpy(dz, s->dz.data(), 4 * (size_t)s->Klive);
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

extern "C" int cg_set_tuning(cg_sim* s, int snapshot_interval, int cluster_size)
{
    if (!s) return CG_EINVAL;
    int shift = s->snap_shift, pref = s->cluster_pref;
    if (snapshot_interval) {
        if (snapshot_interval != 1 && snapshot_interval != 2 && snapshot_interval != 4 && snapshot_interval != 8) return CG_EINVAL;
        shift = snapshot_interval == 1 ? 0 : snapshot_interval == 2 ? 1 : snapshot_interval == 4 ? 2 : 3;
        s->snap_auto = false;
    }
    if (cluster_size) {
        if (cluster_size != -1 && (cluster_size < 1 || cluster_size > CG_MAX_CLUSTER || (cluster_size & (cluster_size - 1)))) return CG_EINVAL;
        pref = cluster_size == -1 ? 0 : cluster_size;
    }
    CK(cudaStreamSynchronize(s->stream));
    const int old_pref = s->cluster_pref;
    s->snap_shift = shift; s->cluster_pref = pref;
    if (pref != old_pref) {
        const int rc = choose_launch(s, 0, 0);
        if (rc != CG_OK) { s->cluster_pref = old_pref; choose_launch(s, 0, 0); return rc; }
    }
    return CG_OK;
}

extern "C" int cg_get_tuning(cg_sim* s, int* snapshot_interval, int* cluster_size)
{
    if (!s) return CG_EINVAL;
    if (snapshot_interval) *snapshot_interval = 1 << s->snap_shift;
    if (cluster_size) *cluster_size = s->cluster;
    return CG_OK;
}

extern "C" int cg_get_exchange_cycles(cg_sim* s, uint64_t* cycles6)
{
    if (!s || !cycles6) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    for (int k = 0; k < 6; ++k) cycles6[k] = c.cyc_x[k];
    return CG_OK;
}

extern "C" int cg_get_kernel(cg_sim* s, int* kind)
{
    if (!s || !kind) return CG_EINVAL;
    *kind = s->single ? 1 : 0;
    return CG_OK;
}

extern "C" int cg_get_labels_per_thread(cg_sim* s, int* labels_per_thread)
{
    if (!s || !labels_per_thread) return CG_EINVAL;
    *labels_per_thread = s->pl > 0 ? s->lpt : 0;
    return CG_OK;
}

extern "C" int cg_set_phase_timers(cg_sim* s, int on)
{
    if (!s) return CG_EINVAL;
    s->timers = on != 0;
    return CG_OK;
}

extern "C" int cg_get_phase_cycles(cg_sim* s, uint64_t* total, uint64_t* wait, uint64_t* update,
                                   uint64_t* propose, uint64_t* warps, int reset)
{
    if (!s) return CG_EINVAL;
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    if (total) *total = c.cyc_total;
    if (wait) *wait = c.cyc_wait;
    if (update) *update = c.cyc_update;
    if (propose) *propose = c.cyc_propose;
    if (warps) *warps = c.cyc_warps;
    if (reset) {
        c.cyc_total = c.cyc_wait = c.cyc_update = c.cyc_propose = c.cyc_warps = 0;
        for (int k = 0; k < 6; ++k) c.cyc_x[k] = 0;
        CK(cudaMemcpyAsync(s->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s->stream));
        CK(cudaStreamSynchronize(s->stream));
    }
    return CG_OK;
}

extern "C" int cg_bench_l2(size_t bytes, int reps, int trials, int mode, int ctas_per_sm, int threads, int vec_bytes,
                           double* gbps)
{
    cg_sim* s = nullptr;
    if (!gbps || bytes < 4096 || (bytes & 31) || reps < 1 || trials < 1 || mode < 0 || mode > 2 || ctas_per_sm < 1
        || ctas_per_sm > 16 || threads < 32 || threads > 1024 || (threads & 31) || (vec_bytes != 16 && vec_bytes != 32))
        return CG_EINVAL;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* buf = nullptr;
    CK(cudaMalloc(&buf, bytes + 256));
    struct Free { void* p; ~Free() { cudaFree(p); } } fr{buf};
    CK(cudaMemset(buf, 0, bytes + 256));
    EventPair ev;
    CK(cudaEventCreate(&ev.a)); CK(cudaEventCreate(&ev.b));
    const size_t nvec = bytes / (size_t)vec_bytes;
    const int grid = (int)std::max<size_t>(1, std::min<size_t>((nvec + threads - 1) / threads, (size_t)sms * ctas_per_sm));
    double* sink = buf + bytes / 8;
    auto launch = [&](int r) {
        if (vec_bytes == 16) cg_l2_probe<16><<<grid, threads>>>(buf, nvec, r, mode, sink);
        else cg_l2_probe<32><<<grid, threads>>>(buf, nvec, r, mode, sink);
    };
    launch(2);                                             // warm-up
    float best = 1e30f;
    for (int t = 0; t < trials; ++t) {
        CK(cudaEventRecord(ev.a));
        launch(reps);
        CK(cudaEventRecord(ev.b));
        CK(cudaEventSynchronize(ev.b));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ev.a, ev.b));
        best = std::min(best, ms);
    }
    CK(cudaGetLastError());
    const double moved = (mode == 0 ? 2.0 : 1.0) * (double)bytes * (double)reps;
    *gbps = moved / ((double)best * 1e-3) / 1e9;
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
        case CG_EDEVICE: return "the persistent kernel abandoned a launch (see cg_last_error)";
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

// ---- cg_get_dos_noalloc: the same histogram without any allocation -------------------------------------
// For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops): the scratch bins of
// cg_dos live in a file-scope device array of CG_DOS_NOALLOC_MAX_BINS + 1 counters (64 KiB + 8 B, held by
// every GPU that loads the library until exit).  In host code the array's name is only a host-side stand-in
// for the symbol: its device address is taken once per device, with that device current, by
// cudaGetSymbolAddress, and only that pointer is ever given to a kernel or a copy.
static __device__ __align__(256) unsigned long long cg_dos_static_bins[CG_DOS_NOALLOC_MAX_BINS + 1];

#define CG_MAX_DEVICES 64
static unsigned long long* g_dos_bins_addr[CG_MAX_DEVICES];      // device address of the array on device d, once known
static std::mutex g_dos_bins_mutex;

// device address of cg_dos_static_bins on the sim's device, which must be the current one
static int dos_static_bins(cg_sim* s, unsigned long long** out)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev != s->device || dev < 0 || dev >= CG_MAX_DEVICES) {
        s->err = "cg_get_dos_noalloc: the sim's device must be the current device";
        return CG_EINVAL;
    }
    std::lock_guard<std::mutex> lock(g_dos_bins_mutex);
    if (!g_dos_bins_addr[dev]) {
        void* ptr = nullptr;
        CK(cudaGetSymbolAddress(&ptr, cg_dos_static_bins));
        if (!ptr) { s->err = "cudaGetSymbolAddress returned a null address"; return CG_ECUDA; }
        g_dos_bins_addr[dev] = (unsigned long long*)ptr;
    }
    *out = g_dos_bins_addr[dev];
    return CG_OK;
}

extern "C" int cg_get_dos_noalloc(cg_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside)
{
    if (!s || !hist || !(width > 0.0) || nbins == 0) return CG_EINVAL;
    if (nbins > CG_DOS_NOALLOC_MAX_BINS) {
        char buf[160];
        snprintf(buf, sizeof buf, "cg_get_dos_noalloc: nbins = %u exceeds the static scratch of %u bins "
                                  "(use cg_get_dos)", nbins, (unsigned)CG_DOS_NOALLOC_MAX_BINS);
        s->err = buf;
        return CG_EINVAL;
    }
    CgCtl c;
    int rc = read_ctl(s, &c);
    if (rc != CG_OK) return rc;
    unsigned long long* bins = nullptr;
    if ((rc = dos_static_bins(s, &bins)) != CG_OK) return rc;
    // the array keeps the counts of the last call: everything this call reads back starts at zero
    CK(cudaMemsetAsync(bins, 0, 8 * ((size_t)nbins + 1), s->stream));
    const u32 nsh = nbins <= 8192 ? nbins : 0;
    const unsigned grid = std::max(1u, std::min((s->N + 2047) / 2048, 148u * 4));
    cg_dos<<<grid, 256, 4 * (size_t)nsh, s->stream>>>(s->d_eps[c.cur % CG_RING], s->N, lo, width, nbins, nsh, bins);
    CK(cudaGetLastError());
    unsigned long long out_of_range = 0;
    CK(cudaMemcpyAsync(hist, bins, 8 * (size_t)nbins, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaMemcpyAsync(&out_of_range, bins + nbins, 8, cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (outside) *outside = out_of_range;
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
    if (first > have || count > have - first) return CG_EINVAL;
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
