/*
 * cg_oracle.c — CPU ORACLE (TEST INFRASTRUCTURE ONLY; see cg_oracle.h).
 *
 * Plain, slow, serial C in fp64, written from /root/reference/PAPER.md
 * (arXiv 1407.5026).  Every function cites the passage it follows; step
 * numbers O1..O10 are the bit-level readings listed in DESIGN.md.
 * The same code runs the 2D lattice of the paper and its
 * cubic 3D extension (reading G22 in DESIGN.md): a 2D lattice
 * is the case Lz = 1 of an Lz x L x L torus, site s = (z L + y) L + x, so every
 * loop below runs over (z, y, x) and visits the sites of a 2D lattice in the
 * order s = y L + x.
 * Build: gcc -O2 -ffp-contract=off (no fast-math).  OpenMP is used ONLY for
 * the one-time O(N^2) full-sum of eps over the outer site index s; the sum
 * over t stays sequential (O6), and the Monte Carlo loop is single-threaded.
 */
#include "cg_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

struct cgo_sim {
    /* parameters */
    int      L;        /* lattice side                                          */
    int      Lz;       /* 1: the paper's 2D L x L lattice; L: cubic 3D */
    uint32_t N;        /* Lz * L * L sites, s = (z L + y) L + x                 */
    double   W, xi, T, E;
    uint64_t seed;
    uint32_t M;
    /* state */
    double*  phi;      /* N   random potentials              */
    int8_t*  n;        /* N   occupations                    */
    double*  eps;      /* N   single-particle energies       */
    /* translation-invariant tables */
    double*  invr;     /* Lz*L*L 1/r for offset ((dz mod Lz),(dy mod L),(dx mod L)) */
    int64_t  K;        /* number of allowed displacements                  */
    int32_t* ddz;      /* K   (all 0 in 2D)                                */
    int32_t* ddy;      /* K                                                */
    int32_t* ddx;      /* K                                                */
    double*  invr_k;   /* K   1/r of displacement k                        */
    double*  cdf;      /* K   tower                          */
    double   S;        /* sum_k w_k                                        */
    double   Gamma;    /* N * S                              */
    /* counters */
    uint64_t attempts;     /* next unused attempt index = attempts consumed */
    uint64_t last_end;     /* attempts consumed at the previous executed hop */
    uint64_t hops;
    double   t_stoch;      /* O11: sum of the Gaussian increments of step 3c */
    uint64_t iterations;   /* PR iterations a width-M PR run would need     */
    uint64_t proposals_evaluated; /* iterations * M                         */
    int64_t  dP;
    uint64_t near_ties;
    uint64_t exp_evals;
    double   update_seconds;
    double   fixed_A;      /* <0: physical acceptance                       */
    /* hop log */
    int       log_on;
    uint64_t  log_len, log_cap;
    uint64_t* log_a;
    uint32_t* log_i;
    uint32_t* log_j;
};

/* ---------------------------------------------------------------- O1 ---- */
/* Philox4x32-10, Salmon, Moraes, Dror, Shaw, SC'11:
 * ten rounds of  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with the key bumped by the Weyl constants between rounds. */
void cgo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_domain(const cgo_sim* s, uint64_t index, uint32_t domain, uint32_t w[4])
{
    /* O1: key = seed, counter = (index lo, index hi, domain, 0);
     * domain 0 = KMC attempts, 1 = phi, 2 = occupation keys. */
    uint32_t ctr[4] = { (uint32_t)index, (uint32_t)(index >> 32), domain, 0u };
    uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    cgo_philox4x32_10(ctr, key, w);
}

/* ---------------------------------------------------------------- G7 ---- */
void cgo_pr_split(uint64_t m, uint32_t M, uint64_t* p, uint32_t* q)
{
    /* "M = 12, p = 2, q = 5" for the 17th serial attempt. */
    *p = (m - 1) / M + 1;
    *q = (uint32_t)((m - 1) % M) + 1;
}

/* ------------------------------------------------------------ geometry -- */
/* Minimum image of a lattice offset, components in (-L/2, L/2];
 * the tie at exactly L/2 resolves to +L/2 (reading G3). */
static int min_image(int d, int L)
{
    d = ((d % L) + L) % L;
    if (d > L / 2) d -= L;
    return d;
}

/* Periodic wrap of a coordinate difference or sum, valid for -L <= v < 2L. */
static int wrap(int v, int L)
{
    if (v < 0) v += L;
    else if (v >= L) v -= L;
    return v;
}

/* Coordinates of site a = (z L + y) L + x (z = 0 in 2D). */
static inline void site_zyx(const cgo_sim* s, uint32_t a, int* z, int* y, int* x)
{
    uint32_t L = (uint32_t)s->L;
    *x = (int)(a % L);
    *y = (int)((a / L) % L);
    *z = (int)(a / (L * L));
}

/* 1/r_ab under minimum image for sites a, b; 0 on the diagonal (O4). */
static inline double invr_sites(const cgo_sim* s, uint32_t a, uint32_t b)
{
    int L = s->L, Lz = s->Lz;
    int za, ya, xa, zb, yb, xb;
    site_zyx(s, a, &za, &ya, &xa);
    site_zyx(s, b, &zb, &yb, &xb);
    return s->invr[((size_t)wrap(za - zb, Lz) * (size_t)L + (size_t)wrap(ya - yb, L)) * (size_t)L
                   + (size_t)wrap(xa - xb, L)];
}

double cgo_invr_sites(const cgo_sim* s, uint32_t a, uint32_t b) { return invr_sites(s, a, b); }

/* ---------------------------------------------------------------- O4/O5 - */
struct disp { int64_t r2; int32_t dz, dy, dx; };

static int disp_cmp(const void* pa, const void* pb)
{
    const struct disp* a = (const struct disp*)pa;
    const struct disp* b = (const struct disp*)pb;
    if (a->r2 != b->r2) return a->r2 < b->r2 ? -1 : 1;
    if (a->dz != b->dz) return a->dz < b->dz ? -1 : 1;
    if (a->dy != b->dy) return a->dy < b->dy ? -1 : 1;
    if (a->dx != b->dx) return a->dx < b->dx ? -1 : 1;
    return 0;
}

static int build_tables(cgo_sim* s)
{
    int L = s->L, Lz = s->Lz, h = L / 2;
    /* 1/r for every offset of the torus, r = minimum-image Euclidean distance
     * in lattice units; no image sums. */
    s->invr = (double*)malloc(sizeof(double) * (size_t)Lz * (size_t)L * (size_t)L);
    if (!s->invr) return CGO_ENOMEM;
    for (int c = 0; c < Lz; ++c)
        for (int a = 0; a < L; ++a)
            for (int b = 0; b < L; ++b) {
                int dc = min_image(c, Lz), da = min_image(a, L), db = min_image(b, L);
                int64_t r2 = (int64_t)dc * dc + (int64_t)da * da + (int64_t)db * db;
                s->invr[((size_t)c * L + a) * L + b] = (r2 == 0) ? 0.0 : 1.0 / sqrt((double)r2);
            }
    /* Allowed hops: 0 < r <= L/2 ("We do not allow hops larger than L/2",
     * PAPER.md:90), each ordered pair once: components in (-L/2, L/2]
     * (dz = 0 only, in 2D). */
    int zlo = (Lz == 1) ? 0 : -h + 1, zhi = (Lz == 1) ? 0 : h;
    size_t cap = (size_t)Lz * (size_t)L * (size_t)L;
    struct disp* d = (struct disp*)malloc(sizeof(struct disp) * cap);
    if (!d) return CGO_ENOMEM;
    int64_t K = 0;
    for (int dz = zlo; dz <= zhi; ++dz)
        for (int dy = -h + 1; dy <= h; ++dy)
            for (int dx = -h + 1; dx <= h; ++dx) {
                int64_t r2 = (int64_t)dz * dz + (int64_t)dy * dy + (int64_t)dx * dx;
                if (r2 > 0 && r2 <= (int64_t)h * h) {
                    d[K].r2 = r2; d[K].dz = dz; d[K].dy = dy; d[K].dx = dx; ++K;
                }
            }
    qsort(d, (size_t)K, sizeof(struct disp), disp_cmp);     /* order (r2, dz, dy, dx): G12, G22 */
    s->K = K;
    s->ddz = (int32_t*)malloc(sizeof(int32_t) * (size_t)K);
    s->ddy = (int32_t*)malloc(sizeof(int32_t) * (size_t)K);
    s->ddx = (int32_t*)malloc(sizeof(int32_t) * (size_t)K);
    s->invr_k = (double*)malloc(sizeof(double) * (size_t)K);
    s->cdf = (double*)malloc(sizeof(double) * (size_t)K);
    if (!s->ddz || !s->ddy || !s->ddx || !s->invr_k || !s->cdf) { free(d); return CGO_ENOMEM; }
    /* Tower of Gamma^T_ij = exp(-2 r_ij / xi): running sum in
     * list order, normalised by the total. */
    double run = 0.0;
    for (int64_t k = 0; k < K; ++k) {
        s->ddz[k] = d[k].dz; s->ddy[k] = d[k].dy; s->ddx[k] = d[k].dx;
        double r = sqrt((double)d[k].r2);
        s->invr_k[k] = 1.0 / r;
        double t = -2.0 * r;
        double w = exp(t / s->xi);
        run = run + w;
        s->cdf[k] = run;
    }
    s->S = run;
    for (int64_t k = 0; k < K; ++k) s->cdf[k] = s->cdf[k] / s->S;
    s->cdf[K - 1] = 1.0;
    /* On a lattice Gamma^T depends on r only, so Gamma = N sum_j Gamma^T_ij
     * (PAPER.md:80). */
    s->Gamma = (double)s->N * s->S;
    free(d);
    return CGO_OK;
}

/* ---------------------------------------------------------------- O6 ---- */
/* eps_i = phi_i + sum_{j != i} (n_j - nu)/r_ij, nu = 1/2,
 * summed in index order j = 0..N-1. */
static void full_sum_eps(const cgo_sim* s, double* out)
{
    int L = s->L, Lz = s->Lz;
    int64_t N = (int64_t)s->N;
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < N; ++a) {
        int za, ya, xa;
        site_zyx(s, (uint32_t)a, &za, &ya, &xa);
        double e = s->phi[a];
        for (int zb = 0; zb < Lz; ++zb)
            for (int yb = 0; yb < L; ++yb) {             /* b = (zb*L + yb)*L + xb ascending */
                const double* row = s->invr + ((size_t)wrap(za - zb, Lz) * (size_t)L
                                               + (size_t)wrap(ya - yb, L)) * (size_t)L;
                const int8_t* nb = s->n + ((size_t)zb * (size_t)L + (size_t)yb) * (size_t)L;
                for (int xb = 0; xb < L; ++xb) {
                    if (zb == za && yb == ya && xb == xa) continue;
                    e += ((double)nb[xb] - 0.5) * row[wrap(xa - xb, L)];
                }
            }
        out[a] = e;
    }
}

/* ---------------------------------------------------------------- O2/O3 - */
struct keyed { uint64_t key; uint32_t site; };

static int keyed_cmp(const void* pa, const void* pb)
{
    const struct keyed* a = (const struct keyed*)pa;
    const struct keyed* b = (const struct keyed*)pb;
    if (a->key != b->key) return a->key < b->key ? -1 : 1;
    if (a->site != b->site) return a->site < b->site ? -1 : 1;
    return 0;
}

static int build_disorder_and_occupations(cgo_sim* s)
{
    uint32_t N = s->N;
    /* phi_i uniform of full width W centred on 0 (reading G2). */
    for (uint32_t a = 0; a < N; ++a) {
        uint32_t w[4];
        philox_domain(s, a, 1u, w);
        uint64_t bits = (((uint64_t)w[0] << 32) | (uint64_t)w[1]) >> 11;   /* 53 bits */
        double u = (double)bits * 0x1p-53;
        s->phi[a] = (u - 0.5) * s->W;
    }
    /* "random initial configuration" with exactly nu*N electrons
     * (PAPER.md:52, 84): the N/2 sites with the smallest random keys. */
    struct keyed* ks = (struct keyed*)malloc(sizeof(struct keyed) * N);
    if (!ks) return CGO_ENOMEM;
    for (uint32_t a = 0; a < N; ++a) {
        uint32_t w[4];
        philox_domain(s, a, 2u, w);
        ks[a].key = ((uint64_t)w[0] << 32) | (uint64_t)w[1];
        ks[a].site = a;
    }
    qsort(ks, N, sizeof(struct keyed), keyed_cmp);
    memset(s->n, 0, N);
    for (uint32_t r = 0; r < N / 2; ++r) s->n[ks[r].site] = 1;
    free(ks);
    return CGO_OK;
}

/* ------------------------------------------------------------------------ */
static int init_lattice(cgo_sim** out, int dim, int L, double W, double xi, double T, double E,
                        uint64_t seed, uint32_t M)
{
    if (!out) return CGO_EINVAL;
    *out = NULL;
    if (L < 2 || (L % 2) != 0 || L > (dim == 3 ? 256 : 4096)) return CGO_EINVAL;
    if (!(xi > 0.0) || !(T > 0.0) || !(W >= 0.0) || M < 1 || !isfinite(E)) return CGO_EINVAL;
    cgo_sim* s = (cgo_sim*)calloc(1, sizeof(cgo_sim));
    if (!s) return CGO_ENOMEM;
    s->L = L; s->Lz = (dim == 3) ? L : 1;
    s->N = (uint32_t)s->Lz * (uint32_t)L * (uint32_t)L;
    s->W = W; s->xi = xi; s->T = T; s->E = E; s->seed = seed; s->M = M;
    s->fixed_A = -1.0;
    s->phi = (double*)malloc(sizeof(double) * s->N);
    s->eps = (double*)malloc(sizeof(double) * s->N);
    s->n = (int8_t*)malloc(s->N);
    int rc = (!s->phi || !s->eps || !s->n) ? CGO_ENOMEM : CGO_OK;
    if (rc == CGO_OK) rc = build_tables(s);
    if (rc == CGO_OK) rc = build_disorder_and_occupations(s);
    if (rc != CGO_OK) { cgo_free(s); return rc; }
    full_sum_eps(s, s->eps);
    *out = s;
    return CGO_OK;
}

int cgo_init(cgo_sim** out, int L, double W, double xi, double T, double E,
             uint64_t seed, uint32_t M)
{
    return init_lattice(out, 2, L, W, xi, T, E, seed, M);
}

/* The cubic lattice the paper names as the natural extension (PAPER.md:118
 * "significantly more advantageous in 3D than in 2D", "easily
 * extended to higher dimensions"): N = L^3, same Hamiltonian, rates and
 * algorithm, field along x (reading G22). */
int cgo_init3(cgo_sim** out, int L, double W, double xi, double T, double E,
              uint64_t seed, uint32_t M)
{
    return init_lattice(out, 3, L, W, xi, T, E, seed, M);
}

void cgo_free(cgo_sim* s)
{
    if (!s) return;
    free(s->phi); free(s->eps); free(s->n); free(s->invr);
    free(s->ddz); free(s->ddy); free(s->ddx); free(s->invr_k); free(s->cdf);
    free(s->log_a); free(s->log_i); free(s->log_j);
    free(s);
}

/* ---------------------------------------------------------------- O7 ---- */
/* One attempt of the mixed algorithm (steps 1-2 of PAPER.md:73-74):
 * propose (i,j) with probability Gamma^T_ij / Gamma by tower sampling —
 * i uniform over the N sites (G5), displacement k with probability w_k / S —
 * and decode the acceptance uniform.  State is not touched. */
static void decode_attempt(const cgo_sim* s, uint64_t a, uint32_t* i, uint32_t* j, int64_t* k,
                           double* u_d, double* u_a)
{
    uint32_t w[4];
    philox_domain(s, a, 0u, w);
    *i = (uint32_t)(((uint64_t)w[0] * (uint64_t)s->N) >> 32);
    uint64_t bd = ((uint64_t)w[1] << 11) | (uint64_t)(w[2] >> 21);          /* 43 bits */
    uint64_t ba = ((uint64_t)(w[2] & 0x1FFFFFu) << 32) | (uint64_t)w[3];    /* 53 bits */
    *u_d = (double)bd * 0x1p-43;
    *u_a = (double)ba * 0x1p-53;
    int64_t kk = 0;
    while (!(*u_d < s->cdf[kk])) ++kk;          /* tower sampling [7]: smallest k with u < cdf_k */
    *k = kk;
    int L = s->L, Lz = s->Lz;
    int zi, yi, xi_;
    site_zyx(s, *i, &zi, &yi, &xi_);
    int zj = wrap(zi + s->ddz[kk], Lz), yj = wrap(yi + s->ddy[kk], L), xj = wrap(xi_ + s->ddx[kk], L);
    *j = ((uint32_t)zj * (uint32_t)L + (uint32_t)yj) * (uint32_t)L + (uint32_t)xj;
}

int cgo_decode_attempt(const cgo_sim* s, uint64_t a, uint32_t* i, uint32_t* j, int64_t* k,
                       double* u_d, double* u_a)
{
    if (!s) return CGO_EINVAL;
    uint32_t ii, jj; int64_t kk; double ud, ua;
    decode_attempt(s, a, &ii, &jj, &kk, &ud, &ua);
    if (i) *i = ii;
    if (j) *j = jj;
    if (k) *k = kk;
    if (u_d) *u_d = ud;
    if (u_a) *u_a = ua;
    return CGO_OK;
}

/* Acceptance with probability Gamma^A_ij = theta_ij min[1, exp(-dH_ij/T)]
 * (Eq.(2)), dH_ij = eps_j - eps_i - 1/r_ij - E dx_ij
 * (PAPER.md:63). */
static int accept_attempt(cgo_sim* s, uint32_t i, uint32_t j, int64_t k, double u_a)
{
    if (s->fixed_A >= 0.0) return u_a < s->fixed_A;      /* PAPER.md:41 pin: constant acceptance */
    if (s->n[i] != 1) return 0;                          /* theta_ij = delta(n_i,1) delta(n_j,0) */
    if (s->n[j] != 0) return 0;
    double dE = s->eps[j] - s->eps[i];
    dE = dE - s->invr_k[k];
    double field = s->E * (double)s->ddx[k];
    dE = dE - field;
    if (dE <= 0.0) return 1;
    double x = (-dE) / s->T;
    double p = exp(x);
    s->exp_evals++;
    /* O10 near-tie certificate: decisions are libm-independent unless u_a lies
     * within a few ulp of exp(x). */
    if (fabs(u_a - p) <= 0x1p-50 * p) s->near_ties++;
    return u_a < p;
}

/* ---------------------------------------------------------------- O8 ---- */
static double now_seconds(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

/* Step 3a-3b: execute i->j, dP += dx_ij, and add
 * 1/r_lj - 1/r_li to eps_l for every l; with 1/r_ll := 0 this gives
 * +1/r_ij at l=i and -1/r_ij at l=j as the paper lists (reading G1). */
static void execute_hop(cgo_sim* s, uint32_t i, uint32_t j)
{
    int L = s->L, Lz = s->Lz;
    s->n[i] = 0;
    s->n[j] = 1;
    int zi, yi, xi_, zj, yj, xj;
    site_zyx(s, i, &zi, &yi, &xi_);
    site_zyx(s, j, &zj, &yj, &xj);
    s->dP += (int64_t)min_image(xj - xi_, L);
    double t0 = now_seconds();
    for (int z = 0; z < Lz; ++z)
        for (int y = 0; y < L; ++y) {
            const double* row_j = s->invr + ((size_t)wrap(z - zj, Lz) * (size_t)L + (size_t)wrap(y - yj, L)) * (size_t)L;
            const double* row_i = s->invr + ((size_t)wrap(z - zi, Lz) * (size_t)L + (size_t)wrap(y - yi, L)) * (size_t)L;
            double* e = s->eps + ((size_t)z * (size_t)L + (size_t)y) * (size_t)L;
            for (int x = 0; x < L; ++x) {
                double d = row_j[wrap(x - xj, L)] - row_i[wrap(x - xi_, L)];
                e[x] = e[x] + d;
            }
        }
    s->update_seconds += now_seconds() - t0;
}

static int log_push(cgo_sim* s, uint64_t a, uint32_t i, uint32_t j)
{
    if (s->log_len == s->log_cap) {
        uint64_t cap = s->log_cap ? 2 * s->log_cap : 1024;
        uint64_t* na = (uint64_t*)realloc(s->log_a, sizeof(uint64_t) * cap);
        if (!na) return CGO_ENOMEM;
        s->log_a = na;
        uint32_t* ni = (uint32_t*)realloc(s->log_i, sizeof(uint32_t) * cap);
        if (!ni) return CGO_ENOMEM;
        s->log_i = ni;
        uint32_t* nj = (uint32_t*)realloc(s->log_j, sizeof(uint32_t) * cap);
        if (!nj) return CGO_ENOMEM;
        s->log_j = nj;
        s->log_cap = cap;
    }
    s->log_a[s->log_len] = a; s->log_i[s->log_len] = i; s->log_j[s->log_len] = j;
    s->log_len++;
    return CGO_OK;
}

/* --------------------------------------------------------------- O11 ---- */
/* Standard normal deviate of executed hop h (0-based), Box-Muller transform of
 * one Philox block of domain 3, counter = (h lo, h hi, 3, 0):
 *   u1 = (((w0:w1) >> 11) + 1) * 2^-53  in (0,1],  u2 = ((w2:w3) >> 11) * 2^-53  in [0,1),
 *   z  = sqrt(-2 ln u1) * cos(2 pi u2).
 * The paper only asks for "a Gaussian distribution"; the
 * transform and the word use are reading G19. */
static double normal_of_hop(const cgo_sim* s, uint64_t h)
{
    uint32_t w[4];
    philox_domain(s, h, 3u, w);
    uint64_t a = (((uint64_t)w[0] << 32) | (uint64_t)w[1]) >> 11;
    uint64_t b = (((uint64_t)w[2] << 32) | (uint64_t)w[3]) >> 11;
    double u1 = (double)(a + 1u) * 0x1p-53;
    double u2 = (double)b * 0x1p-53;
    double rad = sqrt(-2.0 * log(u1));
    double ang = 6.283185307179586476925286766559 * u2;
    return rad * cos(ang);
}

double cgo_normal_of_hop(const cgo_sim* s, uint64_t h) { return s ? normal_of_hop(s, h) : 0.0; }

/* Step 3c: "Increment the time by a random dt sampled from a
 * Gaussian distribution of mean m/Gamma and standard deviation sqrt(m)/Gamma",
 * m = attempts consumed since the previous executed hop (reading G7). */
static double gaussian_dt(const cgo_sim* s, uint64_t h, uint64_t m)
{
    double mean = (double)m / s->Gamma;
    double sd   = sqrt((double)m) / s->Gamma;
    return mean + sd * normal_of_hop(s, h);
}

/* Bookkeeping common to physical and scripted hops: m attempts were consumed
 * since the previous executed hop; a width-M PR run needs p = ceil(m/M)
 * iterations for them (G7, G8) and evaluates p*M proposals (G18). */
static int account_hop(cgo_sim* s, uint64_t a, uint32_t i, uint32_t j)
{
    uint64_t m = (a + 1) - s->last_end, p; uint32_t q;
    cgo_pr_split(m, s->M, &p, &q);
    s->iterations += p;
    s->proposals_evaluated += p * (uint64_t)s->M;
    s->last_end = a + 1;
    s->t_stoch += gaussian_dt(s, s->hops, m);            /* O11, hop index 0-based */
    s->hops++;
    return s->log_on ? log_push(s, a, i, j) : CGO_OK;
}

/* The serial rejection algorithm for the mixed chain
 * (PAPER.md:71): attempt after attempt on the current state; the first
 * accepted proposal is executed. */
int cgo_run(cgo_sim* s, uint64_t n_hops)
{
    if (!s) return CGO_EINVAL;
    uint64_t target = s->hops + n_hops;
    while (s->hops < target) {
        uint64_t a = s->attempts;
        uint32_t i, j; int64_t k; double u_d, u_a;
        decode_attempt(s, a, &i, &j, &k, &u_d, &u_a);
        int ok = accept_attempt(s, i, j, k, u_a);
        s->attempts = a + 1;
        if (ok) {
            if (s->fixed_A < 0.0) execute_hop(s, i, j);
            int rc = account_hop(s, a, i, j);
            if (rc != CGO_OK) return rc;
        }
    }
    return CGO_OK;
}

int cgo_apply_hops(cgo_sim* s, uint64_t count, const uint32_t* i, const uint32_t* j)
{
    if (!s || (count && (!i || !j))) return CGO_EINVAL;
    for (uint64_t h = 0; h < count; ++h) {
        if (i[h] >= s->N || j[h] >= s->N || i[h] == j[h]) return CGO_EINVAL;
        if (s->n[i[h]] != 1 || s->n[j[h]] != 0) return CGO_EINVAL;
        execute_hop(s, i[h], j[h]);
        s->hops++;
    }
    return CGO_OK;
}

/* ---------------------------------------------------------------- O9 ---- */
int cgo_get_state(const cgo_sim* s, int8_t* n, double* eps, double* t_tau0, int64_t* dP)
{
    if (!s) return CGO_EINVAL;
    if (n) memcpy(n, s->n, s->N);
    if (eps) memcpy(eps, s->eps, sizeof(double) * s->N);
    /* deterministic increment dt = m/Gamma per executed hop,
     * i.e. t = (attempts consumed)/Gamma. */
    if (t_tau0) *t_tau0 = (double)s->attempts / s->Gamma;
    if (dP) *dP = s->dP;
    return CGO_OK;
}

int cgo_get_counters(const cgo_sim* s, uint64_t* attempts, uint64_t* proposals_evaluated,
                     uint64_t* iterations, uint64_t* hops)
{
    if (!s) return CGO_EINVAL;
    if (attempts) *attempts = s->attempts;
    if (proposals_evaluated) *proposals_evaluated = s->proposals_evaluated;
    if (iterations) *iterations = s->iterations;
    if (hops) *hops = s->hops;
    return CGO_OK;
}

int cgo_enable_hop_log(cgo_sim* s, int enable)
{
    if (!s) return CGO_EINVAL;
    s->log_on = enable ? 1 : 0;
    return CGO_OK;
}

int cgo_get_hops(const cgo_sim* s, uint64_t first, uint64_t count,
                 uint64_t* attempt, uint32_t* i, uint32_t* j)
{
    if (!s || first + count > s->log_len) return CGO_EINVAL;
    for (uint64_t h = 0; h < count; ++h) {
        if (attempt) attempt[h] = s->log_a[first + h];
        if (i) i[h] = s->log_i[first + h];
        if (j) j[h] = s->log_j[first + h];
    }
    return CGO_OK;
}

int cgo_recompute_eps(const cgo_sim* s, double* eps_out, double* max_abs_dev)
{
    if (!s) return CGO_EINVAL;
    double* tmp = (double*)malloc(sizeof(double) * s->N);
    if (!tmp) return CGO_ENOMEM;
    full_sum_eps(s, tmp);
    double dev = 0.0;
    for (uint32_t a = 0; a < s->N; ++a) {
        double d = fabs(tmp[a] - s->eps[a]);
        if (d > dev) dev = d;
    }
    if (eps_out) memcpy(eps_out, tmp, sizeof(double) * s->N);
    if (max_abs_dev) *max_abs_dev = dev;
    free(tmp);
    return CGO_OK;
}

int64_t cgo_num_displacements(const cgo_sim* s) { return s ? s->K : -1; }

int cgo_get_tables(const cgo_sim* s, int32_t* dy, int32_t* dx, double* cdf, double* invr_k,
                   double* S, double* Gamma)
{
    if (!s) return CGO_EINVAL;
    size_t K = (size_t)s->K;
    if (dy) memcpy(dy, s->ddy, sizeof(int32_t) * K);
    if (dx) memcpy(dx, s->ddx, sizeof(int32_t) * K);
    if (cdf) memcpy(cdf, s->cdf, sizeof(double) * K);
    if (invr_k) memcpy(invr_k, s->invr_k, sizeof(double) * K);
    if (S) *S = s->S;
    if (Gamma) *Gamma = s->Gamma;
    return CGO_OK;
}

int cgo_get_dz(const cgo_sim* s, int32_t* dz)
{
    if (!s || !dz) return CGO_EINVAL;
    memcpy(dz, s->ddz, sizeof(int32_t) * (size_t)s->K);
    return CGO_OK;
}

int cgo_dimension(const cgo_sim* s) { return s ? (s->Lz == 1 ? 2 : 3) : 0; }

int cgo_get_phi(const cgo_sim* s, double* phi)
{
    if (!s || !phi) return CGO_EINVAL;
    memcpy(phi, s->phi, sizeof(double) * s->N);
    return CGO_OK;
}

int cgo_set_state(cgo_sim* s, const int8_t* n, uint64_t next_attempt)
{
    if (!s || !n) return CGO_EINVAL;
    uint64_t sum = 0;
    for (uint32_t a = 0; a < s->N; ++a) {
        if (n[a] != 0 && n[a] != 1) return CGO_EINVAL;
        sum += (uint64_t)n[a];
    }
    if (sum != s->N / 2) return CGO_EINVAL;              /* sum_i n_i = nu N */
    memcpy(s->n, n, s->N);
    full_sum_eps(s, s->eps);
    s->attempts = next_attempt;
    s->last_end = next_attempt;
    return CGO_OK;
}

int cgo_set_phi(cgo_sim* s, const double* phi)
{
    if (!s || !phi) return CGO_EINVAL;
    memcpy(s->phi, phi, sizeof(double) * s->N);
    full_sum_eps(s, s->eps);
    return CGO_OK;
}

int cgo_set_fixed_A(cgo_sim* s, double A)
{
    if (!s) return CGO_EINVAL;
    s->fixed_A = A;
    return CGO_OK;
}

uint64_t cgo_near_ties(const cgo_sim* s) { return s ? s->near_ties : 0; }
uint64_t cgo_exp_evaluations(const cgo_sim* s) { return s ? s->exp_evals : 0; }
double   cgo_update_seconds(const cgo_sim* s) { return s ? s->update_seconds : 0.0; }

/* ------------------------------------------------- observables (O11-O14) -- */
/* O11: elapsed time with the stochastic increment of step 3c. */
int cgo_get_time_stochastic(const cgo_sim* s, double* t_tau0)
{
    if (!s || !t_tau0) return CGO_EINVAL;
    *t_tau0 = s->t_stoch;
    return CGO_OK;
}

/* O12: single-particle density of states: histogram of the eps_k
 * with bin size width, bin b = [lo + b*width, lo + (b+1)*width), as counts;
 * g(eps) = hist / (N * width).  Sites outside [lo, lo + nbins*width) are
 * counted in *outside. */
int cgo_dos(const cgo_sim* s, double lo, double width, uint32_t nbins, uint64_t* hist, uint64_t* outside)
{
    if (!s || !hist || !(width > 0.0) || nbins == 0) return CGO_EINVAL;
    uint64_t out = 0;
    for (uint32_t b = 0; b < nbins; ++b) hist[b] = 0;
    for (uint32_t k = 0; k < s->N; ++k) {
        double x = floor((s->eps[k] - lo) / width);
        if (x >= 0.0 && x < (double)nbins) hist[(uint32_t)x]++;
        else out++;
    }
    if (outside) *outside = out;
    return CGO_OK;
}

/* O13: polarisation against time (Fig.3 inset): after logged
 * hop h, t_h = (a_h + 1)/Gamma (deterministic increment) and
 * P_h - P_start = sum of dx over logged hops 0..h. */
int cgo_get_series(const cgo_sim* s, uint64_t first, uint64_t count, double* t, int64_t* P)
{
    if (!s || first + count > s->log_len) return CGO_EINVAL;
    int64_t acc = 0;
    for (uint64_t h = 0; h < first + count; ++h) {
        int xi_ = (int)(s->log_i[h] % (uint32_t)s->L), xj = (int)(s->log_j[h] % (uint32_t)s->L);
        acc += (int64_t)min_image(xj - xi_, s->L);
        if (h >= first) {
            if (t) t[h - first] = (double)(s->log_a[h] + 1u) / s->Gamma;
            if (P) P[h - first] = acc;
        }
    }
    return CGO_OK;
}

/* O14: stationary conductivity estimate sigma0 = P/(N E t) (Eq.(3)
 * PAPER.md:65), P = dP accumulated since t = 0, t deterministic. */
int cgo_sigma0(const cgo_sim* s, double* sigma0)
{
    if (!s || !sigma0 || s->E == 0.0 || s->attempts == 0) return CGO_EINVAL;
    double t = (double)s->attempts / s->Gamma;
    *sigma0 = (double)s->dP / (((double)s->N * s->E) * t);
    return CGO_OK;
}
