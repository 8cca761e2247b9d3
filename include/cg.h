/*
 * cg.h — C ABI of libcg.so: the B200-native (sm_100a) hot path of the parallel
 * kinetic Monte Carlo for Coulomb glasses of Ferrero, Kolton and Palassini
 * (arXiv 1407.5026; citations are lines of /root/reference/PAPER.md).
 *
 * What the library computes: the "mixed PR algorithm" of PAPER.md:71-78 on an
 * L x L periodic lattice at half filling (cg_init), or on the L x L x L cubic
 * lattice the paper names as its natural extension (cg_init3) —
 *   1. M labelled proposals per iteration, each (i, j) drawn with probability
 *      Gamma^T_ij / Gamma, Gamma^T_ij = exp(-2 r_ij / xi)
 *   2. each accepted with probability theta_ij min[1, exp(-dH_ij/T)],
 *      dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
 *   3. the lowest accepting label q is executed, dP += dx_ij, every local
 *      energy gets eps_l += 1/r_lj - 1/r_li, time advances by m/Gamma
 *
 * looped on the device without a host round trip per hop.  The random stream is
 * Philox4x32-10 keyed by (seed, global attempt index), so the
 * sequence of executed hops is identical to that of the serial mixed algorithm
 * ("mathematically equivalent") and does not depend on M or on the
 * launch shape.  DESIGN.md lists every reading of the paper this relies on.
 *
 * Conventions: site s = y*L + x (row-major, x = field direction; 3D: s = (z*L + y)*L + x),
 * sites, labels and attempt indices 0-based.  All pointers are HOST pointers unless the name
 * starts with dev_.  All functions return CG_OK (0) or a negative CG_E* code;
 * none throws, aborts or prints.  A sim is not thread-safe; distinct sims are
 * independent.  There is no CPU fallback: without a CUDA device every compute
 * entry point fails with CG_ECUDA.
 */
#ifndef CG_H_
#define CG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cg_sim cg_sim; /* opaque; owned by the library, released by cg_free */

#define CG_OK            0
#define CG_EINVAL       (-1)  /* bad argument (NULL, odd L, T<=0, xi<=0, M==0, range) */
#define CG_ENOMEM       (-2)  /* host or device allocation failed / workspace too small */
#define CG_ECUDA        (-3)  /* a CUDA call failed; text kept for cg_last_error       */
#define CG_EUNSUPPORTED (-4)  /* valid problem the sm_100a path does not cover:
                                 L not a power of two, L > 1024 (3D: L > 64),
                                 M > 2^27, or a live tower longer than 65535
                                 displacements (very large xi)                     */
#define CG_EDEVICE      (-5)  /* the device-side watchdog abandoned a launch: some
                                 wait inside the persistent kernel took longer than
                                 10 s (CG_WATCHDOG_MS in the environment of cg_init
                                 overrides; 0 = never).  Reported by the next call
                                 that synchronises; the state is undefined until
                                 cg_set_state.  Never seen in a correct build: it
                                 turns a would-be hang into an error              */

/* Problem statement.  L: lattice side, N = L*L sites, a power
 * of two in [4, 1024]; W: full width of the uniform disorder, phi_i in [-W/2, W/2);
 * xi: localisation length; T: temperature (k_B = 1); E: field along +x in the
 * sense of dH = ... - E dx; seed: Philox key; M >= 1: logical PR width (labels per
 * iteration; may exceed the number of resident threads).
 * Filling nu = 1/2 and the hop cut-off r <= L/2 are fixed.
 * cg_init allocates its own device memory on the current device and uses the
 * legacy default stream.  On failure *out is NULL. */
int cg_init(cg_sim** out, int L, double W, double xi, double T, double E,
            uint64_t seed, uint32_t M);

/* The same on the cubic lattice, N = L^3 sites, L a power of two in [4, 64]
 * ("significantly more advantageous in 3D than in 2D", PAPER.md:122
 * "easily extended to higher dimensions"): displacements (dz, dy, dx) with
 * 0 < r <= L/2 in the order (r^2, dz, dy, dx), field along x.  Every other call
 * takes either kind of sim. */
int cg_init3(cg_sim** out, int L, double W, double xi, double T, double E,
             uint64_t seed, uint32_t M);

/* Same, for callers that own device memory (e.g. a torch uint8 tensor) and a
 * stream: dev_workspace must hold cg_workspace_bytes(L, M) bytes, be 256-byte
 * aligned and outlive the sim; cuda_stream is a cudaStream_t (NULL = default). */
size_t cg_workspace_bytes(int L, uint32_t M);
int cg_init_ws(cg_sim** out, int L, double W, double xi, double T, double E,
               uint64_t seed, uint32_t M,
               void* dev_workspace, size_t bytes, void* cuda_stream);
size_t cg_workspace_bytes3(int L, uint32_t M);
int cg_init3_ws(cg_sim** out, int L, double W, double xi, double T, double E,
                uint64_t seed, uint32_t M,
                void* dev_workspace, size_t bytes, void* cuda_stream);

/* Advance exactly n_accepted_hops executed hops (not iterations) of the chain.
 * One persistent cooperative kernel per 2^30 hops; asynchronous on the sim's stream.
 * cg_run(a); cg_run(b) is the same chain as cg_run(a+b). */
int cg_run(cg_sim* s, uint64_t n_accepted_hops);

/* Replica packing (averaging many samples at intermediate L is the
 * recommended use): advance EACH of the n_sims independent sims by
 * n_accepted_hops executed hops in ONE persistent launch, every sim on its own
 * CTAs side by side; each chain is exactly the one cg_run would produce.
 * sims[] is a host array of distinct sims that share device, stream and launch
 * shape (either all single-CTA sims - 512 threads, any number of them, one CTA each -
 * or 544 threads with the same register tiling and label caching: true for
 * sims of equal L whose M fits their CTAs; see cg_get_launch / cg_set_launch); the sum of
 * their CTA counts must fit on the device at once, else CG_EUNSUPPORTED; clusters are not used.
 * Asynchronous on that stream; the array is not referenced after the call. */
int cg_run_many(cg_sim* const* sims, int n_sims, uint64_t n_accepted_hops);

/* Synchronises the stream and copies out: occupations n[N] in {0,1}
 * (PAPER.md:52), local energies eps[N], elapsed time
 * t = attempts_consumed / Gamma in units of tau0 (deterministic increment
 * m/Gamma, with m = (p-1)M + q), and the net
 * charge displacement dP = sum of dx over executed hops.
 * Any pointer may be NULL. */
int cg_get_state(cg_sim* s, int8_t* n, double* eps, double* t_tau0, int64_t* dP);

/* Restore a state previously read with cg_get_state / cg_get_counters
 * (checkpoint): n[N] with sum N/2, eps[N], attempts consumed, hops, dP.
 * iterations / proposals counters restart from zero. */
int cg_set_state(cg_sim* s, const int8_t* n, const double* eps,
                 uint64_t attempts, uint64_t hops, int64_t dP);

/* Counters: attempts consumed (sum of m), proposals evaluated (M per
 * iteration), PR iterations, executed hops.  Synchronises the stream. */
int cg_get_counters(cg_sim* s, uint64_t* attempts, uint64_t* proposals_evaluated,
                    uint64_t* iterations, uint64_t* hops);

/* Hop log: (attempt index, i, j) of executed hops.  cg_enable_hop_log reserves
 * room for `capacity` hops counted from the current hop; dev_buf (may be NULL:
 * the library allocates) must hold 16*capacity bytes.  cg_get_hops copies hops
 * [first, first+count) of the log (indices relative to the enabling point);
 * CG_EINVAL outside the logged range, and after cg_apply_hops (scripted hops are
 * not logged) until the log is enabled again. */
int cg_enable_hop_log(cg_sim* s, uint64_t capacity, void* dev_buf, size_t bytes);
int cg_get_hops(cg_sim* s, uint64_t first, uint64_t count,
                uint64_t* attempt, uint32_t* i, uint32_t* j);

/* ---- Observables: read-only device passes, outside the hot loop; each
 * synchronises the sim's stream.  All output pointers are HOST pointers owned by the caller.
 *
 * cg_get_time_stochastic: elapsed time with the random increment of step 3c:
 *   per executed hop h, dt_h = m_h/Gamma + (sqrt(m_h)/Gamma) z_h, m_h = attempts consumed
 *   since the previous executed hop, z_h a standard normal deviate (Box-Muller of the Philox
 *   block counter = (h lo, h hi, 3, 0), h = 0-based count of executed hops; G19).
 *   m_h comes from the hop log, so the log must be enabled and must hold EVERY hop executed by
 *   cg_run since it was enabled (CG_EINVAL otherwise, also after scripted hops of cg_apply_hops, which
 *   are not logged, until the log is enabled again or cg_set_state is called); time before the enabling point enters
 *   with the deterministic increment.  Summed in a fixed tree order (bit-reproducible).
 * cg_get_normals: z[k] = z_{first_hop + k}, k < count (parity hook for the above).
 * cg_get_dos: density of states as bin counts of eps: hist[b] = #{k : lo + b*width
 *   <= eps_k < lo + (b+1)*width}, b < nbins <= 2^24, width > 0; *outside (may be NULL) = sites in
 *   no bin.  g(eps) = hist / (N * width).
 * cg_get_series: polarisation against time (Fig.3 inset) over logged hops
 *   [first, first+count): t[k] = (a_h + 1)/Gamma (deterministic increment) and
 *   P[k] = sum of dx over logged hops 0..h, h = first + k; t or P may be NULL.
 *   Needs the complete hop log like cg_get_time_stochastic.
 * cg_get_sigma0: sigma0 = dP/(N E t), t deterministic (Eq.(3));
 *   CG_EINVAL for E = 0 or t = 0. */
int cg_get_time_stochastic(cg_sim* s, double* t_tau0);
int cg_get_normals(cg_sim* s, uint64_t first_hop, uint64_t count, double* z);
int cg_get_dos(cg_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside);
int cg_get_series(cg_sim* s, uint64_t first, uint64_t count, double* t, int64_t* P);

/* cg_get_dos_noalloc: cg_get_dos for callers that must not allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same result, same kernel;
 * the only difference is where the kernel's scratch bins live: in a file-scope device array of the
 * library (CG_DOS_NOALLOC_MAX_BINS + 1 64-bit counters = 64 KiB + 8 B of device memory, held by every
 * GPU that loads libcg.so until the process exits) instead of a cudaMalloc'ed buffer.  The call performs
 * no cudaMalloc / cudaFree and no allocating library call; hist and outside are HOST pointers owned by
 * the caller and written directly.
 *   nbins > CG_DOS_NOALLOC_MAX_BINS -> CG_EINVAL (cg_last_error names the limit; use cg_get_dos).
 *   The sim's device must be the current device (CG_EINVAL otherwise): the array's device address is
 *   looked up once per device with that device current.
 *   ALL calls on one GPU share the one array, which keeps the counts of the previous call; each call
 *   clears the part it uses first.  Calls that overlap on the GPU (sims on different streams, several
 *   host threads) race on it and return garbage: serialise them.  Synchronises the sim's stream. */
#define CG_DOS_NOALLOC_MAX_BINS 8192u
int cg_get_dos_noalloc(cg_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside);
int cg_get_sigma0(cg_sim* s, double* sigma0);

/* Recompute eps from its definition eps_i = phi_i + sum_{j!=i}(n_j - 1/2)/r_ij
 * on the device and return max_i |eps_i - eps_i^incremental|. */
int cg_recompute_eps(cg_sim* s, double* max_abs_dev);

/* Step a6 alone: execute `count` scripted hops i[h] -> j[h] (occupations,
 * dP and the O(N) update of PAPER.md:77; no acceptance test, no time) in one
 * launch of the update kernel.  Used for parity of the update against the
 * oracle and for its bandwidth measurement.  Every hop must satisfy theta_ij
 * (n_i = 1, n_j = 0) at its turn: otherwise CG_EINVAL and nothing is changed.
 * ms (may be NULL) receives the device time of the launch measured with CUDA
 * events on the sim's stream.
 * Two kernels compute the same sums (bit-identical): "staged" keeps whole lattice rows of
 * eps in shared memory and brings the two table rows every lattice row needs per hop in
 * with bulk asynchronous copies (cp.async.bulk + mbarrier), three hops ahead; "gathers"
 * keeps eps in registers and reads the table with per-site loads.  cg_set_update_kernel:
 * 0 = automatic (the faster one as measured on B200: gathers), 1 = gathers, 2 = staged
 * (cg_apply_hops then returns CG_EUNSUPPORTED when the rows do not fit shared memory or
 * L < 32). */
int cg_apply_hops(cg_sim* s, uint64_t count, const uint32_t* i, const uint32_t* j, float* ms);
int cg_set_update_kernel(cg_sim* s, int kind);

/* Diagnostics of the one-time set-up (step a0): translation-invariant tables
 * (PAPER.md:80).  K = number of displacements with 0 < r <= L/2 in the order
 * (r^2, dy, dx); K_live = length of the prefix whose tower value is < 1 plus
 * one (later entries can never be drawn by a uniform u < 1). */
int cg_get_table_sizes(cg_sim* s, int64_t* K, int64_t* K_live);
int cg_get_tables(cg_sim* s, int32_t* dy, int32_t* dx, double* cdf, double* invr_k, /* K_live each */
                  double* S, double* Gamma);
int cg_get_table_dz(cg_sim* s, int32_t* dz /* K_live; all 0 on the 2D lattice */);
int cg_get_phi(cg_sim* s, double* phi /* N */);

/* Launch shape of the persistent kernel: n_ctas in [1, co-resident maximum] (a multiple
 * of the cluster size), threads in {256, 544, 608, 1024} = 32 x (5, 14, 16 or 29 worker
 * warps + 3 service warps); 0 keeps the heuristic.  Results never depend on it.
 * (1, 512) is the single-CTA kernel: 512 worker threads, eps and occupations in shared
 * memory, two CTA barriers per iteration - for sims with M <= 512 labels and N <= 8192
 * sites (CG_EINVAL otherwise); (1, 1024) is the same kernel with 1024 threads when
 * 512 < M <= 1024 and N <= 8192 (otherwise the dataflow shape of that size); (1, 512) with
 * M > 512 or N > 8192 is the variant with 2, 4 or 8 labels per thread (M <= 4096,
 * N <= 16384: a lattice of L = 128 on one SM, for replica packing).  The heuristic
 * picks the single-CTA kernel whenever M <= 1024, N <= 1024 and no cluster size was asked
 * for.  cg_get_launch reports the shape in use, cg_get_kernel which kernel it belongs to. */
int cg_set_launch(cg_sim* s, int n_ctas, int threads);
int cg_get_launch(cg_sim* s, int* n_ctas, int* threads, int* smem_bytes);
/* Which kernel cg_run launches in the shape in use: *kind = 0 the dataflow kernel cg_pr_persistent, 1 the
 * single-CTA kernel cg_pr_single (512 threads for M <= 512, 1024 threads for M <= 1024). */
int cg_get_kernel(cg_sim* s, int* kind);

/* Tuning that never changes results.  snapshot_interval H in {1, 2, 4, 8} (default: 8 for N >= 2^18
 * sites, else 2): the
 * eps slabs, kept current in registers after every hop, are written through to memory
 * every H hops (deferred update; PAPER.md:77, 106 W_U); cluster_size in {1, 2, 4, 8, 16}:
 * CTAs per thread-block cluster, whose members post their results into each other's
 * shared memory instead of through L2; -1 = automatic (the default: clusters of up to 16
 * when the whole sim fits 96 CTAs, pairs when it wants every SM - clusters of 8 and 16 leave
 * SMs of a B200 unused).  0 leaves a value as it is.  A new cluster size re-derives the
 * launch shape (CG_EUNSUPPORTED if the device cannot co-schedule it).  cg_set_launch with an
 * explicit CTA count keeps the largest cluster size that divides it; cg_get_tuning reports
 * the cluster size in use.  cg_run_many launches without clusters. */
int cg_set_tuning(cg_sim* s, int snapshot_interval, int cluster_size);
/* How the M labels of an iteration are held in the launch shape in use: *labels_per_thread =
 * K >= 1: every worker thread keeps K proposals decoded (attempts a, a + P, ..., a + (K-1) P with P = CTAs x
 * worker threads >= M / K) and only re-tests them in every iteration (K = 1 whenever M <= P; K <= 8, 544-thread
 * shape, while the extra slots fit shared memory); 0: M is larger than that and every label is decoded and
 * tested from scratch in every iteration (time linear in M).  Results never depend on it. */
int cg_get_labels_per_thread(cg_sim* s, int* labels_per_thread);
int cg_get_tuning(cg_sim* s, int* snapshot_interval, int* cluster_size);

/* The paper's split of the time per hop into rejection and update time (PAPER.md:106:
 * "the sum of two main contributions: the rejection time W_R ... and the update time W_U"),
 * measured inside the persistent kernel that runs, in SM clock cycles, accumulated over
 * cg_run calls: *total = cycles CTA 0 spent in the kernel; the other three are SUMS over
 * the *warps worker warps of CTA 0 of the cycles a warp spent (propose) consuming the
 * previous outcome, testing its proposals and handing in its lowest accept, (update)
 * updating its part of the eps slab, (wait) waiting for the outcome of the iteration.
 * Per warp, propose + update + wait = total up to start-up; W_U per hop = update / warps /
 * hops, W_R per hop = (propose + wait) / warps / hops.  reset != 0 zeroes the counters.
 * The timers cost a few per cent (three clock reads per warp and iteration), so they are off
 * by default: cg_set_phase_timers(s, 1) makes the following cg_run calls use the timed build
 * of the same kernel (544-thread launch shapes only; otherwise nothing is recorded). */
int cg_set_phase_timers(cg_sim* s, int on);
/* The select side of W_R (step 3) from the same timed build: cycles6[0..4] = SUMS over the exchange
 * warps of all CTAs of the cycles spent (0) waiting until the slowest consumer of the CTA has released the
 * descriptor slot, (1) at the gate on published eps snapshots, (2) at scan position 0: waiting for the CTA's own
 * workers, (3) scanning the posts of the CTAs in label order, (4) deciding and publishing the outcome;
 * cycles6[5] = exchange warps that contributed (CTAs x launches).  Reset together with cg_get_phase_cycles. */
int cg_get_exchange_cycles(cg_sim* s, uint64_t* cycles6);
int cg_get_phase_cycles(cg_sim* s, uint64_t* total, uint64_t* wait, uint64_t* update,
                        uint64_t* propose, uint64_t* warps, int reset);

/* L2 roofline probe: one kernel, `ctas_per_sm` CTAs of `threads`
 * threads per SM, L1-bypassing accesses of vec_bytes (16 or 32) over a resident buffer of
 * `bytes`, `reps` passes inside the launch; mode 0 read-modify-write, 1 read only, 2 write
 * only.  Returns GB/s (mode 0 counts read + written bytes) of the best of `trials` launches. */
int cg_bench_l2(size_t bytes, int reps, int trials, int mode, int ctas_per_sm, int threads,
                int vec_bytes, double* gbps);

void cg_free(cg_sim* s);
const char* cg_strerror(int code);
const char* cg_last_error(cg_sim* s); /* text of the last CUDA failure, "" if none */

#ifdef __cplusplus
}
#endif
#endif
