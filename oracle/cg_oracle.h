/*
 * cg_oracle.h — CPU ORACLE for the Coulomb-glass kinetic Monte Carlo of
 * Ferrero, Kolton, Palassini (arXiv 1407.5026).  TEST INFRASTRUCTURE ONLY.
 *
 * This is the plain serial "mixed" rejection algorithm driven by
 * a counter-based random stream indexed by the global attempt index.  The
 * paper states that the parallel-rejection (PR) algorithm "is mathematically
 * equivalent to the serial mixed algorithm", so the serial
 * chain IS the definition of what the GPU path must compute.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call anything in oracle/.
 * It shares no code with paper_1407_5026_b200/ (the CUDA path) and neither
 * imports the other.
 *
 * Parity pins (tests/test_oracle_*.py, `-m "not gpu"`): see DESIGN.md §Oracle.
 * Unpinned: the steady-state statistical physics of the paper (A≈0.03T,
 * DOS slope, Efros–Shklovskii fits) — "parity unpinned" for those; they are
 * out of scope of the hot path.
 *
 * Conventions: site s = y*L + x, x = field direction;
 * labels and attempt indices are 0-based.
 */
#ifndef CG_ORACLE_H_
#define CG_ORACLE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cgo_sim cgo_sim;

#define CGO_OK       0
#define CGO_EINVAL  (-1)
#define CGO_ENOMEM  (-2)

/* Philox4x32-10 (Salmon et al. SC'11, PAPER.md:138 ref [9]).  O1. */
void cgo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* PR bookkeeping (Fig.1(a), PAPER.md:78 step 3c, reading G7):
 * the m-th serial attempt (1-based) since the previous executed hop falls in
 * parallel iteration p (1-based) with label q (1-based): m = (p-1)*M + q. */
void cgo_pr_split(uint64_t m, uint32_t M, uint64_t* p, uint32_t* q);

/* Problem statement: L x L torus, half filling,
 * phi ~ U[-W/2, W/2), localisation length xi, temperature T, field E along x,
 * Philox seed, logical PR width M (only enters the iteration bookkeeping). */
int  cgo_init(cgo_sim** out, int L, double W, double xi, double T, double E,
              uint64_t seed, uint32_t M);
/* Cubic 3D lattice, N = L^3, site s = (z L + y) L + x, field along x — the
 * extension the paper names; everything else as cgo_init.
 * Every other call works on either kind of sim (N is then L^3). */
int  cgo_init3(cgo_sim** out, int L, double W, double xi, double T, double E,
               uint64_t seed, uint32_t M);
void cgo_free(cgo_sim* s);

/* Advance exactly n_hops executed hops of the serial mixed algorithm. */
int  cgo_run(cgo_sim* s, uint64_t n_hops);

/* Outputs: occupations n[N], local energies eps[N],
 * t = attempts/Gamma in tau0 (PAPER.md:84 deterministic increment),
 * dP = sum of dx over executed hops.  Any pointer may be NULL. */
int  cgo_get_state(const cgo_sim* s, int8_t* n, double* eps, double* t_tau0, int64_t* dP);
int  cgo_get_counters(const cgo_sim* s, uint64_t* attempts, uint64_t* proposals_evaluated,
                      uint64_t* iterations, uint64_t* hops);

/* Hop log: (attempt index, i, j) of executed hops [first, first+count). */
int  cgo_enable_hop_log(cgo_sim* s, int enable);
int  cgo_get_hops(const cgo_sim* s, uint64_t first, uint64_t count,
                  uint64_t* attempt, uint32_t* i, uint32_t* j);

/* eps recomputed from its definition vs the incremental value. */
int  cgo_recompute_eps(const cgo_sim* s, double* eps_out /*N or NULL*/, double* max_abs_dev);

/* Tables: K displacements sorted by (r2, dy, dx); cdf; 1/r_k; Gamma.  O4/O5. */
int64_t cgo_num_displacements(const cgo_sim* s);
int  cgo_get_tables(const cgo_sim* s, int32_t* dy, int32_t* dx, double* cdf, double* invr_k,
                    double* S, double* Gamma);
int  cgo_get_dz(const cgo_sim* s, int32_t* dz /* K; all 0 in 2D; list order is (r2, dz, dy, dx) */);
int  cgo_dimension(const cgo_sim* s);   /* 2 or 3 */
/* 1/r under minimum image between sites a and b (0 for a==b). */
double cgo_invr_sites(const cgo_sim* s, uint32_t a, uint32_t b);

/* Disorder phi[N]. */
int  cgo_get_phi(const cgo_sim* s, double* phi);

/* Decode attempt a into its proposal and uniforms without touching state (O7). */
int  cgo_decode_attempt(const cgo_sim* s, uint64_t a, uint32_t* i, uint32_t* j, int64_t* k,
                        double* u_d, double* u_a);

/* Test hooks. */
int  cgo_set_state(cgo_sim* s, const int8_t* n, uint64_t next_attempt); /* n: N entries, sum N/2; eps recomputed */
int  cgo_set_phi(cgo_sim* s, const double* phi);                        /* eps recomputed */
int  cgo_set_fixed_A(cgo_sim* s, double A); /* A>=0: accept iff u_a < A, state untouched (PAPER.md:41 pin); A<0: physical */
int  cgo_apply_hops(cgo_sim* s, uint64_t count, const uint32_t* i, const uint32_t* j); /* execute scripted hops (no test) */
uint64_t cgo_near_ties(const cgo_sim* s);   /* O10 certificate counter */
uint64_t cgo_exp_evaluations(const cgo_sim* s);
double   cgo_update_seconds(const cgo_sim* s); /* wall time spent in the O(N) update (W_U) */


/* Observables.
 * O11 stochastic time: per executed hop h (0-based count since cgo_init),
 *     dt = m/Gamma + (sqrt(m)/Gamma) * z_h  (PAPER.md:78 step 3c), z_h standard
 *     normal by Box-Muller from Philox domain 3 (reading G19), summed in hop order.
 * O12 density of states as bin counts.
 * O13 polarisation series (t_h, P_h) over the hop log.
 * O14 sigma0 = dP/(N E t). */
double cgo_normal_of_hop(const cgo_sim* s, uint64_t h);
int  cgo_get_time_stochastic(const cgo_sim* s, double* t_tau0);
int  cgo_dos(const cgo_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside);
int  cgo_get_series(const cgo_sim* s, uint64_t first, uint64_t count, double* t, int64_t* P);
int  cgo_sigma0(const cgo_sim* s, double* sigma0);

#ifdef __cplusplus
}
#endif
#endif
