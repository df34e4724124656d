/*
 * oracle/jump_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU implementation of the hot path of the Velocity-Jumps
 * (JUMP) integrator of arXiv 2412.15073, written from /root/reference/PAPER.md
 * ("P:Lnnn" = line nnn of that file) and the readings R-n listed in DESIGN.md.
 * It shares no code with the CUDA path (paper_2412_15073_b200/csrc): only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.
 *
 * What is computed, in the paper's order and notation:
 *   - Langevin BAOAB splitting                    P:L112-125, eq. (2)
 *   - force decomposition grad U = F0 + sum F_ij
 *   - general jump mechanism (6),(7), Theta, f_eta P:L84-98, pairwise P:L338-346
 *   - BPS mechanism (4),(5) for Lennard-Jones
 *   - Poisson thinning, Algorithm 4 (step C)
 *   - ring technique
 *   - Algorithm 5 (step J, BPS)
 *   - rejection sampler for G~
 *   - C'J'AOAJ'C' scheme
 *   - JUMP-RESPA / BAOAB-RESPA
 *   - JUMP-RESPA1 / BAOAB-RESPA1 (three levels) with the reciprocal Ewald sum as the slow
 *     many-body force F_{0,1}                      P:L145, P:L509-511, P:L325 (R-21)
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): Philox known-answer
 * vectors; closed forms of Theta and of the G~ CDF/mean; chi end conditions and
 * short+long = unsplit; finite differences of U; brute-force O(N^2) sums;
 * stationarity identity of (6),(7); eps=inf == BPS; eps->0 mean drift == -F/m;
 * thinning invariance under inflated bounds, under the two list policies and under
 * the two forms of the bound of Algorithm 4 (R-11); OU stationary variance; BAOAB
 * energy conservation / reversibility; 2-body Boltzmann histogram (with and without
 * acceleration); rows and cell universe against an independent restatement of their
 * rules; LJ bound over a range of sigma; degenerate cases.
 * "Parity unpinned" by the paper (fixed by DESIGN.md readings only):
 * the formula of chi, the bound recipe L, r_A and r_M, the list policy (skin, order,
 * cell universe), the G~ proposal details, the Philox stream layout, k_cut of the
 * reciprocal sum and the outermost step ratio of RESPA1 (R-21).  The reciprocal sum
 * itself is pinned (Madelung constants, finite differences, a closed form on one molecule).
 *
 * List policies (orc_params.list_policy): 1 = R-10c, the contract of the CUDA path: rings
 * [r_c-h, r_A), [r_A, r_M), [r_M, r_long) by CURRENT distance, candidates from two
 * skin-padded rows and from the cell universe; 0 = R-10 (round 1): rows M, L, V with ring
 * membership by build-time distance.  Both are exact (thinning); the pins run
 * both and compare their accepted jumps.
 *
 * Sign convention (R-4): every "F" here is a GRADIENT piece (grad U = sum F),
 * physical force = -F, exactly as in the paper.
 *
 * Units (R-1): Angstrom, ps, g/mol; energies kcal/mol at the interface;
 * 1 kcal/mol = 418.4 g A^2 mol^-1 ps^-2.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif
/* threads for the loops over n atoms: one per 128 atoms (a 192-atom box on 8 threads spent its
 * time waiting at barriers -- minutes when the host was busy; nothing but the speed depends on it) */
static int orc_threads(int n) {
#ifdef _OPENMP
    int t = n / 128, m = omp_get_max_threads();
    if (t < 1) t = 1;
    return t < m ? t : m;
#else
    (void)n;
    return 1;
#endif
}

#define ORC_KB 1.987204259e-3 /* kcal/mol/K */
#define ORC_COULOMB 332.063713 /* kcal A / (mol e^2) */
#define ORC_KCAL 418.4         /* internal energy units per kcal/mol */
#define ORC_INV_SQRT_2PI 0.39894228040143267794
#define ORC_PI 3.14159265358979323846

/* flags (same meaning as the product's header, restated here on purpose) */
#define ORC_F_COUL_JUMPS 1u
#define ORC_F_LJ_JUMPS 2u
#define ORC_F_EVENT_LOG 4u
#define ORC_F_RESPA_PAPER 8u
#define ORC_F_RESPA_COMPARATOR 16u
#define ORC_F_BJAOAJB 64u /* jump_step runs B J A O A J B instead of C'J' A O A J'C' */
#define ORC_F_COMBINED 128u /* ONE mechanism per pair for the whole long pair gradient, Coulomb + LJ, in step (C'); no (J')
                               (R-22; P:L78-84 a mechanism per force piece F_i, P:L342 F_ij any pair term; needs
                               flags 1 | 2 and list_policy 1) */

/* weight modes of a pair term */
enum { W_NONE = 0, W_SHORT = 1, W_LONG = 2, W_FULL = 3 };

typedef struct {
    int32_t n_atoms, n_inner, eps_mode;
    uint32_t flags;
    int32_t nlist_every;
    int32_t list_policy; /* 0: R-10 (ring rows M, L, V, ring membership by build-time distance); 1: R-10c (rings by
                            current distance, row M, cell universe for the rings L and V) */
    uint64_t seed;
    double box[3];
    double r_short, r_switch, r_mid, r_long, ewald_alpha;
    double dt_fs, gamma_per_ps, temperature_K;
    double eps_jump, skin, cell_edge;
    double r_mid_in; /* R-10c: r_A, inner ring edge (rings [r_c-h, r_A), [r_A, r_M), [r_M, r_long)); <= 0: r_short */
} orc_params;

typedef struct {
    int32_t step, stream, atom, iter;
    int32_t ring;     /* 0 = M, 1 = L, 2 = V (LJ), -1 = clock expired */
    int32_t j;        /* partner (original index) or -1 */
    int32_t accepted; /* 1 if the proposal was accepted */
    int32_t n_gt;     /* attempts of the G~ rejection sampler */
    double T, p, U, gt;
    double margin; /* smallest distance to a discontinuity in this iteration */
} orc_event;

typedef struct {
    int64_t proposals, accepts, gt_attempts, rebuilds, expiries;
    double max_p, max_g_over_L, max_disp, min_margin;
    int64_t min_margin_step;
    /* audit of the list decisions (R-17): smallest |d - window edge| over all candidate pairs of the row builds
     * and smallest distance of an atom to a contract-grid cell face, in A, and the step of that build */
    double min_list_margin;
    int64_t min_list_margin_step;
} orc_stats;

typedef struct {
    orc_params p;
    int n;
    double *x, *xu, *v, *m, *q, *sig, *eps;
    int nb, na;
    int *bij, *aijk;
    double *bk, *br0, *ak, *at0;
    int *excl_ptr, *excl_idx;
    /* derived */
    double kT, beta, dt, alpha, rc, h, rA, rM, rE, skin;
    double *sbm; /* sqrt(beta m_i) in ps/A */
    double *w, w_max; /* mass weights of the skin (R-10c): m_i^-1/2 / mean(m^-1/2) */
    double qmax, eps_max, sig_min, sig_max;
    double GM, GL, G3;   /* sup of the long Coulomb gradient per unit charges over ring 1, 2, 3 (R-7; G3: R-10c only) */
    double GV, GV2, GV3; /* the same for the long LJ gradient with 4 eps = 1 (R-10: GV alone, over the whole shell) */
    int gnx, gny, gnz; /* contract grid for the canonical row order */
    int policy;        /* list policy (orc_params.list_policy) */
    long long last_build; /* step count at the last list build (R-10c schedule) */
    int bound_every;   /* R-11: 1 = B_v and lambda-bar re-evaluated at every proposal, as Algorithm 4 prints them */
    /* R-10c cell universe, built at x_build: atoms of every contract cell (ascending index) and the cell of every atom */
    int *cell_ptr, *cell_atoms, *home, *uni_cnt;
    int uR[3];         /* reach of the universe stencil in cells, per dimension */
    double ureach;     /* r_long + skin */
    /* rows (CSR) built at x_build */
    int *ptrM, *idxM, *ptrL, *idxL, *ptrV, *idxV;
    double *x_build;
    /* gradient pieces, kcal/mol/A */
    double *f_bond, *f_nb, *f0, *f_long;
    int64_t step, outer, outer1;
    /* reciprocal Ewald sum (R-21): half-space vectors n = (nx, ny, nz), k = 2 pi n / box */
    int nk;
    int *kn;
    double *f_slow;
    /* log + stats */
    orc_event *ev;
    int64_t n_ev, cap_ev;
    orc_stats st;
} orc_ctx;

/* ------------------------------------------------------------------ */
/* Philox4x32-10 (R-15).  Salmon et al., SC'11; restated, not copied.  */
/* ------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform in (0,1): (2k+1) 2^-24 with k = top 23 bits, so it has 24 significant bits and is
 * exactly representable in fp32 and fp64 (R-15; the survey's 24-bit variant needs 25 bits) */
double orc_u01(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }

static void chain_block(const orc_ctx *c, int atom, int64_t step, int stream, uint32_t block, uint32_t w[4]) {
    uint32_t ctr[4] = {(uint32_t)atom, (uint32_t)step, (uint32_t)stream, block};
    uint32_t key[2] = {(uint32_t)(c->p.seed & 0xffffffffu), (uint32_t)(c->p.seed >> 32)};
    orc_philox4x32_10(ctr, key, w);
}

/* ------------------------------------------------------------------ */
/* switching function chi (R-3)                                 */
/* ------------------------------------------------------------------ */
void orc_chi(double r, double rc, double h, double *chi, double *dchi) {
    double u = (r - (rc - h)) / h;
    if (u <= 0.0) { *chi = 1.0; *dchi = 0.0; return; }
    if (u >= 1.0) { *chi = 0.0; *dchi = 0.0; return; }
    *chi = 1.0 - u * u * u * (10.0 - 15.0 * u + 6.0 * u * u);
    *dchi = -30.0 * u * u * (1.0 - u) * (1.0 - u) / h;
}

/* ------------------------------------------------------------------ */
/* pair potentials (R-2, R-8): u(r), u'(r)                             */
/* ------------------------------------------------------------------ */
void orc_u_coul(double r, double qq, double alpha, double *u, double *du) {
    /* U_ij = qq erfc(alpha r)/r, qq already holds the Coulomb constant */
    double e = erfc(alpha * r);
    *u = qq * e / r;
    *du = -qq * (e / (r * r) + 2.0 * alpha / sqrt(ORC_PI) * exp(-alpha * alpha * r * r) / r);
}
void orc_u_lj(double r, double sig, double eps, double *u, double *du) {
    /* 4 eps [(s/r)^12 - (s/r)^6]  (P:L441 with the conventional 4, R-8) */
    double s = sig / r, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
    *u = 4.0 * eps * (s12 - s6);
    *du = 4.0 * eps * (-12.0 * s12 + 6.0 * s6) / r;
}
/* radial derivative of w(r) u(r) for the weight modes; 0 beyond r_long */
double orc_weighted_du(int mode, double r, double rc, double h, double rlong, double u, double du) {
    if (mode == W_NONE || r >= rlong) return 0.0;
    if (mode == W_FULL) return du;
    double chi, dchi;
    orc_chi(r, rc, h, &chi, &dchi);
    if (mode == W_SHORT) return chi * du + dchi * u;   /* d/dr [chi u] */
    return (1.0 - chi) * du - dchi * u;                /* d/dr [(1-chi) u] */
}
double orc_weighted_u(int mode, double r, double rc, double h, double rlong, double u) {
    if (mode == W_NONE || r >= rlong) return 0.0;
    if (mode == W_FULL) return u;
    double chi, dchi;
    orc_chi(r, rc, h, &chi, &dchi);
    return mode == W_SHORT ? chi * u : (1.0 - chi) * u;
}

/* ------------------------------------------------------------------ */
/* Theta and the jump mechanism (6),(7)  (R-5)                          */
/* ------------------------------------------------------------------ */
double orc_theta(double eta) {
    /* Theta(eta) = E[(eta+G)_+] = eta Phi(eta) + phi(eta) */
    double Phi = 0.5 * erfc(-eta / sqrt(2.0));
    double phi = ORC_INV_SQRT_2PI * exp(-0.5 * eta * eta);
    return eta * Phi + phi;
}
/* rate: lambda_ij = sqrt(beta)/(eps sqrt(m_i)) |F_ij| Theta(eta);  eps=inf -> (4) */
double orc_jump_rate(double eps, double beta, double sbm, double g, double vn) {
    if (isinf(eps)) return beta * g * (vn > 0.0 ? vn : 0.0);
    return beta * g * orc_theta(eps * sbm * vn) / (eps * sbm);
}
/* kick (P:L344 / eq.(7)); eps=inf -> reflection (5) */
void orc_jump_kick(double eps, double sbm, const double n[3], double gt, double v[3]) {
    double vn = v[0] * n[0] + v[1] * n[1] + v[2] * n[2];
    double amp;
    if (isinf(eps)) amp = 2.0 * vn;
    else {
        double eta = eps * sbm * vn;
        amp = 2.0 * eps / ((1.0 + eps * eps) * sbm) * (eta + gt);
    }
    v[0] -= amp * n[0]; v[1] -= amp * n[1]; v[2] -= amp * n[2];
}

/* ------------------------------------------------------------------ */
/* G~ ~ f_eta by rejection (R-6), proposal family of P:L310.            */
/* One Philox block per attempt, starting at *block.                    */
/* ------------------------------------------------------------------ */
static double upd(double m, double d) { d = fabs(d); return d < m ? d : m; }

double orc_gtilde(const orc_ctx *c, double eta, int atom, int64_t step, int stream,
                  uint32_t *block, int *attempts, double *margin) {
    uint32_t w[4];
    double mg = *margin;
    int it = 0;
    double out = 0.0;
    for (;;) {
        ++it;
        chain_block(c, atom, step, stream, (*block)++, w);
        double u0 = orc_u01(w[0]), u1 = orc_u01(w[1]), u2 = orc_u01(w[2]), u3 = orc_u01(w[3]);
        mg = upd(mg, eta + 2.5); mg = upd(mg, eta + 1.0); mg = upd(mg, eta); /* which proposal family: a decision too */
        if (eta < -2.5) {
            double z = -(log(u0) + log(u1)) / fabs(eta); /* Gamma(2, |eta|) */
            double a = exp(-0.5 * z * z);
            mg = upd(mg, u2 - a);
            if (u2 <= a) { out = z - eta; break; }
        } else if (eta < -1.0) {
            double z = -log(u0) / fabs(eta); /* Exponential(|eta|) */
            double a = z * exp(0.5 * (1.0 - z * z));
            mg = upd(mg, u1 - a);
            if (u1 <= a) { out = z - eta; break; }
        } else if (eta <= 0.0) {
            double z = sqrt(-2.0 * log(u0)); /* Rayleigh */
            double a = exp(eta * z);
            mg = upd(mg, u1 - a);
            if (u1 <= a) { out = z - eta; break; }
        } else {
            double wR = 1.0 / (1.0 + eta * sqrt(2.0 * ORC_PI)); /* Rayleigh-Gaussian mixture */
            mg = upd(mg, u0 - wR);
            if (u0 <= wR) { out = sqrt(-2.0 * log(u1)); break; }
            double y = sqrt(-2.0 * log(u1)) * cos(2.0 * ORC_PI * u2);
            mg = upd(mg, y);
            if (y > 0.0) { out = y; break; }
            mg = upd(mg, y + eta);
            if (y > -eta) {
                double a = (eta + y) / eta;
                mg = upd(mg, u3 - a);
                if (u3 <= a) { out = y; break; }
            }
        }
        if (it >= 64) { out = (eta > 0.0) ? 0.0 : -eta + 1.0; break; } /* P < 1e-11 */
    }
    *attempts = it;
    *margin = mg;
    return out;
}

/* stand-alone entry for the distribution pins */
double orc_gtilde_draw(double eta, uint64_t seed, int atom, int64_t step, int *attempts) {
    orc_ctx c;
    memset(&c, 0, sizeof c);
    c.p.seed = seed;
    uint32_t b = 0;
    double mg = 1e300;
    return orc_gtilde(&c, eta, atom, step, 99, &b, attempts, &mg);
}

/* ------------------------------------------------------------------ */
/* geometry                                                            */
/* ------------------------------------------------------------------ */
static inline void min_image(const orc_ctx *c, const double *xi, const double *xj, double d[3]) {
    for (int k = 0; k < 3; ++k) {
        double dx = xi[k] - xj[k];
        dx -= c->p.box[k] * nearbyint(dx / c->p.box[k]); /* P:L325, minimum image */
        d[k] = dx;
    }
}
static inline double wrap1(double x, double L) {
    x -= L * floor(x / L);
    if (x >= L) x -= L;
    if (x < 0.0) x = 0.0;
    return x;
}
static int is_excluded(const orc_ctx *c, int i, int j) {
    if (!c->excl_ptr) return 0;
    for (int k = c->excl_ptr[i]; k < c->excl_ptr[i + 1]; ++k)
        if (c->excl_idx[k] == j) return 1;
    return 0;
}
static int contract_key(const orc_ctx *c, const double *x) {
    int cc[3], nn[3] = {c->gnx, c->gny, c->gnz};
    for (int k = 0; k < 3; ++k) {
        double xw = wrap1(x[k], c->p.box[k]);
        int ci = (int)floor(xw * ((double)nn[k] / c->p.box[k]));
        if (ci < 0) ci = 0;
        if (ci > nn[k] - 1) ci = nn[k] - 1;
        cc[k] = ci;
    }
    return (cc[2] * c->gny + cc[1]) * c->gnx + cc[0];
}
static double dmax0(double a) { return a > 0.0 ? a : 0.0; }
static int cmp_u64(const void *a, const void *b) {
    uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/*
 * All ordered pairs (i -> j), j != i, not excluded, with minimum-image distance
 * rmin <= d < rmax at positions x, as CSR.  lj_only: keep eps_i eps_j > 0 only.
 * Each row in ascending (contract cell key of j, j) order (R-10).  The search
 * grid below is only an accelerator (checked against brute force in the tests).
 */
static void neighbor_csr_audit(const orc_ctx *c, const double *x, double rmin, double rmax, double hs, int lj_only,
                               int brute, int **ptr_out, int **idx_out, double *edge_margin) {
    /* hs > 0 (R-10c, mass-weighted skin): the window of the pair (i, j) is [rmin - hs (w_i + w_j), rmax + hs (w_i + w_j)) */
    int n = c->n;
    double emin = 1e300;
    int ng[3];
    const double reach = rmax + 2.0 * hs * c->w_max;
    for (int k = 0; k < 3; ++k) {
        ng[k] = (int)floor(c->p.box[k] / reach);
        if (ng[k] < 1) ng[k] = 1;
    }
    int ncell = ng[0] * ng[1] * ng[2];
    int *cell = malloc(sizeof(int) * n), *start = calloc(ncell + 1, sizeof(int)), *order = malloc(sizeof(int) * n);
    int *jkey = malloc(sizeof(int) * n);
    for (int i = 0; i < n; ++i) {
        int cc[3];
        for (int k = 0; k < 3; ++k) {
            double xw = wrap1(x[3 * i + k], c->p.box[k]);
            cc[k] = (int)floor(xw / c->p.box[k] * ng[k]);
            if (cc[k] > ng[k] - 1) cc[k] = ng[k] - 1;
        }
        cell[i] = (cc[2] * ng[1] + cc[1]) * ng[0] + cc[0];
        start[cell[i] + 1]++;
        jkey[i] = contract_key(c, &x[3 * i]);
    }
    for (int k = 0; k < ncell; ++k) start[k + 1] += start[k];
    {
        int *fill = malloc(sizeof(int) * ncell);
        memcpy(fill, start, sizeof(int) * ncell);
        for (int i = 0; i < n; ++i) order[fill[cell[i]]++] = i;
        free(fill);
    }
    int *cnt = calloc(n + 1, sizeof(int));
    uint64_t **rows = malloc(sizeof(uint64_t *) * n);
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(dynamic, 64) reduction(min : emin)
    for (int i = 0; i < n; ++i) {
        int cap = 64, m = 0;
        uint64_t *row = malloc(sizeof(uint64_t) * cap);
        int ci = cell[i];
        int c3[3] = {ci % ng[0], (ci / ng[0]) % ng[1], ci / (ng[0] * ng[1])};
        int lo[3], hi[3];
        for (int k = 0; k < 3; ++k) {
            if (ng[k] < 3 || brute) { lo[k] = 0; hi[k] = ng[k] - 1; }
            else { lo[k] = c3[k] - 1; hi[k] = c3[k] + 1; }
        }
        for (int z = lo[2]; z <= hi[2]; ++z)
            for (int y = lo[1]; y <= hi[1]; ++y)
                for (int xx = lo[0]; xx <= hi[0]; ++xx) {
                    int zc = (z + ng[2]) % ng[2], yc = (y + ng[1]) % ng[1], xc = (xx + ng[0]) % ng[0];
                    int cj = (zc * ng[1] + yc) * ng[0] + xc;
                    for (int s = start[cj]; s < start[cj + 1]; ++s) {
                        int j = order[s];
                        if (j == i) continue;
                        if (lj_only && !(c->eps[i] * c->eps[j] > 0.0)) continue;
                        double d[3];
                        min_image(c, &x[3 * i], &x[3 * j], d);
                        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                        const double sij = hs * (c->w[i] + c->w[j]);
                        const double hi_e = rmax + sij, lo_e = rmin > 0.0 ? dmax0(rmin - sij) : 0.0;
                        const double r2max = hi_e * hi_e, r2min = lo_e * lo_e;
                        if (edge_margin && (fabs(r2 - r2max) < 0.05 || (lo_e > 0.0 && fabs(r2 - r2min) < 0.05)) &&
                            !is_excluded(c, i, j)) { /* audit only: how close is this decision to flipping */
                            double r = sqrt(r2), e = fabs(r - hi_e);
                            if (lo_e > 0.0 && fabs(r - lo_e) < e) e = fabs(r - lo_e);
                            if (e < emin) emin = e;
                        }
                        if (r2 >= r2max || r2 < r2min) continue;
                        if (is_excluded(c, i, j)) continue;
                        if (m == cap) { cap *= 2; row = realloc(row, sizeof(uint64_t) * cap); }
                        row[m++] = ((uint64_t)(uint32_t)jkey[j] << 32) | (uint32_t)j;
                    }
                }
        qsort(row, m, sizeof(uint64_t), cmp_u64);
        rows[i] = row;
        cnt[i + 1] = m;
    }
    for (int i = 0; i < n; ++i) cnt[i + 1] += cnt[i];
    int *idx = malloc(sizeof(int) * (cnt[n] > 0 ? cnt[n] : 1));
    for (int i = 0; i < n; ++i) {
        int m = cnt[i + 1] - cnt[i];
        for (int k = 0; k < m; ++k) idx[cnt[i] + k] = (int)(rows[i][k] & 0xffffffffu);
        free(rows[i]);
    }
    free(rows); free(cell); free(start); free(order); free(jkey);
    *ptr_out = cnt;
    *idx_out = idx;
    if (edge_margin && emin < *edge_margin) *edge_margin = emin;
}
static void neighbor_csr(const orc_ctx *c, const double *x, double rmin, double rmax, int lj_only,
                         int brute, int **ptr_out, int **idx_out) {
    neighbor_csr_audit(c, x, rmin, rmax, 0.0, lj_only, brute, ptr_out, idx_out, NULL);
}

/* exported for the brute-force pin: returns CSR copies */
int orc_neighbors(orc_ctx *c, double rmin, double rmax, int lj_only, int brute, int *ptr, int *idx, int cap) {
    int *p, *ix;
    neighbor_csr(c, c->x, rmin, rmax, lj_only, brute, &p, &ix);
    int tot = p[c->n];
    if (ptr) memcpy(ptr, p, sizeof(int) * (c->n + 1));
    if (idx && tot <= cap) memcpy(idx, ix, sizeof(int) * tot);
    free(p); free(ix);
    return tot;
}

/* ------------------------------------------------------------------ */
/* forces (gradients) and energies                                     */
/* ------------------------------------------------------------------ */
/* gradient w.r.t. x_i of w_C u_C + w_LJ u_LJ for the pair (i,j); returns energy share */
static double pair_gradient(const orc_ctx *c, int i, int j, int wC, int wLJ, double g[3]) {
    double d[3];
    min_image(c, &c->x[3 * i], &c->x[3 * j], d);
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double fr = 0.0, e = 0.0;
    if (wC != W_NONE && c->q[i] * c->q[j] != 0.0) {
        double u, du;
        orc_u_coul(r, ORC_COULOMB * c->q[i] * c->q[j], c->alpha, &u, &du);
        fr += orc_weighted_du(wC, r, c->rc, c->h, c->rE, u, du);
        e += orc_weighted_u(wC, r, c->rc, c->h, c->rE, u);
    }
    if (wLJ != W_NONE && c->eps[i] * c->eps[j] > 0.0) {
        double u, du;
        orc_u_lj(r, sqrt(c->sig[i] * c->sig[j]), sqrt(c->eps[i] * c->eps[j]), &u, &du); /* R-8 */
        fr += orc_weighted_du(wLJ, r, c->rc, c->h, c->rE, u, du);
        e += orc_weighted_u(wLJ, r, c->rc, c->h, c->rE, u);
    }
    for (int k = 0; k < 3; ++k) g[k] = fr * d[k] / r;
    return e;
}

/* out[3n] += sum_j grad_i; returns the pair energy (each pair counted once) */
static double pairs_accumulate(const orc_ctx *c, int wC, int wLJ, int brute, double *out) {
    double rmax = c->rE;
    if ((wC == W_SHORT || wC == W_NONE) && (wLJ == W_SHORT || wLJ == W_NONE)) rmax = c->rc;
    int *ptr, *idx;
    neighbor_csr(c, c->x, 0.0, rmax, 0, brute, &ptr, &idx);
    double etot = 0.0;
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(dynamic, 64) reduction(+ : etot)
    for (int i = 0; i < c->n; ++i) {
        double acc[3] = {0, 0, 0}, e = 0.0;
        for (int k = ptr[i]; k < ptr[i + 1]; ++k) {
            double g[3];
            e += pair_gradient(c, i, idx[k], wC, wLJ, g);
            acc[0] += g[0]; acc[1] += g[1]; acc[2] += g[2];
        }
        out[3 * i] += acc[0]; out[3 * i + 1] += acc[1]; out[3 * i + 2] += acc[2];
        etot += 0.5 * e;
    }
    free(ptr); free(idx);
    return etot;
}

/* harmonic bonds k (r-r0)^2 and angles k (theta-theta0)^2 (R-2); serial, tiny */
static double bonded_accumulate(const orc_ctx *c, double *out) {
    double e = 0.0;
    for (int b = 0; b < c->nb; ++b) {
        int i = c->bij[2 * b], j = c->bij[2 * b + 1];
        double d[3];
        min_image(c, &c->x[3 * i], &c->x[3 * j], d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double dr = r - c->br0[b];
        e += c->bk[b] * dr * dr;
        double f = 2.0 * c->bk[b] * dr / r;
        for (int k = 0; k < 3; ++k) { out[3 * i + k] += f * d[k]; out[3 * j + k] -= f * d[k]; }
    }
    for (int a = 0; a < c->na; ++a) {
        int i = c->aijk[3 * a], j = c->aijk[3 * a + 1], k2 = c->aijk[3 * a + 2]; /* j = vertex */
        double u[3], w[3];
        min_image(c, &c->x[3 * i], &c->x[3 * j], u);
        min_image(c, &c->x[3 * k2], &c->x[3 * j], w);
        double lu = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        double lw = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
        double ct = (u[0] * w[0] + u[1] * w[1] + u[2] * w[2]) / (lu * lw);
        if (ct > 1.0) ct = 1.0;
        if (ct < -1.0) ct = -1.0;
        double th = acos(ct), st = sqrt(1.0 - ct * ct);
        if (st < 1e-12) st = 1e-12;
        double dth = th - c->at0[a];
        e += c->ak[a] * dth * dth;
        double dU = 2.0 * c->ak[a] * dth;
        for (int k = 0; k < 3; ++k) {
            double gi = -dU * (w[k] / lw - ct * u[k] / lu) / (lu * st);
            double gk = -dU * (u[k] / lu - ct * w[k] / lw) / (lw * st);
            out[3 * i + k] += gi;
            out[3 * k2 + k] += gk;
            out[3 * j + k] -= gi + gk;
        }
    }
    return e;
}

/* F0 = bonded + short non-bonded (R-13: LJ tail stays in F0 when LJ jumps are off) */
static void f0_modes(const orc_ctx *c, int *wC, int *wLJ) {
    *wC = W_SHORT;
    *wLJ = (c->p.flags & ORC_F_LJ_JUMPS) ? W_SHORT : W_FULL;
}
static void long_modes(const orc_ctx *c, int *wC, int *wLJ) {
    *wC = W_LONG;
    *wLJ = (c->p.flags & ORC_F_LJ_JUMPS) ? W_LONG : W_NONE;
}
static void compute_f0(orc_ctx *c) {
    int wC, wLJ;
    f0_modes(c, &wC, &wLJ);
    memset(c->f_bond, 0, sizeof(double) * 3 * c->n);
    memset(c->f_nb, 0, sizeof(double) * 3 * c->n);
    bonded_accumulate(c, c->f_bond);
    pairs_accumulate(c, wC, wLJ, 0, c->f_nb);
    for (int k = 0; k < 3 * c->n; ++k) c->f0[k] = c->f_bond[k] + c->f_nb[k];
}
static void compute_bonded_only(orc_ctx *c) {
    memset(c->f_bond, 0, sizeof(double) * 3 * c->n);
    bonded_accumulate(c, c->f_bond);
}
static void compute_long(orc_ctx *c) {
    int wC, wLJ;
    long_modes(c, &wC, &wLJ);
    memset(c->f_long, 0, sizeof(double) * 3 * c->n);
    pairs_accumulate(c, wC, wLJ, 0, c->f_long);
}
static void compute_full(orc_ctx *c, double *out) { /* BAOAB comparator: unsplit to r_long */
    memset(out, 0, sizeof(double) * 3 * c->n);
    bonded_accumulate(c, out);
    pairs_accumulate(c, W_FULL, W_FULL, 0, out);
}

static double slow_accumulate(const orc_ctx *c, double *out);
/* which: 0 F0, 1 full, 2 long, 3 bonded, 4 short non-bonded, 5 slow (reciprocal Ewald + exclusion correction, R-21);
 * brute != 0 -> O(N^2) sweep */
void orc_forces(orc_ctx *c, int which, int brute, double *out) {
    int wC, wLJ;
    memset(out, 0, sizeof(double) * 3 * c->n);
    if (which == 0) { f0_modes(c, &wC, &wLJ); bonded_accumulate(c, out); pairs_accumulate(c, wC, wLJ, brute, out); }
    else if (which == 1) { bonded_accumulate(c, out); pairs_accumulate(c, W_FULL, W_FULL, brute, out); }
    else if (which == 2) { long_modes(c, &wC, &wLJ); pairs_accumulate(c, wC, wLJ, brute, out); }
    else if (which == 3) bonded_accumulate(c, out);
    else if (which == 4) { f0_modes(c, &wC, &wLJ); pairs_accumulate(c, wC, wLJ, brute, out); }
    else if (which == 5) slow_accumulate(c, out);
}
/* which as above; returns potential energy in kcal/mol */
double orc_potential(orc_ctx *c, int which) {
    double *tmp = calloc(3 * c->n, sizeof(double));
    double e = 0.0;
    int wC, wLJ;
    if (which == 0) { f0_modes(c, &wC, &wLJ); e = bonded_accumulate(c, tmp) + pairs_accumulate(c, wC, wLJ, 0, tmp); }
    else if (which == 1) e = bonded_accumulate(c, tmp) + pairs_accumulate(c, W_FULL, W_FULL, 0, tmp);
    else if (which == 2) { long_modes(c, &wC, &wLJ); e = pairs_accumulate(c, wC, wLJ, 0, tmp); }
    else if (which == 3) e = bonded_accumulate(c, tmp);
    else if (which == 4) { f0_modes(c, &wC, &wLJ); e = pairs_accumulate(c, wC, wLJ, 0, tmp); }
    else if (which == 5) e = slow_accumulate(c, tmp);
    free(tmp);
    return e;
}
double orc_kinetic(const orc_ctx *c) {
    double e = 0.0;
    for (int i = 0; i < c->n; ++i)
        e += 0.5 * c->m[i] * (c->v[3 * i] * c->v[3 * i] + c->v[3 * i + 1] * c->v[3 * i + 1] + c->v[3 * i + 2] * c->v[3 * i + 2]);
    return e / ORC_KCAL;
}

/* single-pair long-range gradient pieces used by the jump chains */
static double fij_coul(const orc_ctx *c, int i, int j, double F[3]) {
    double d[3];
    min_image(c, &c->x[3 * i], &c->x[3 * j], d);
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double u, du;
    orc_u_coul(r, ORC_COULOMB * c->q[i] * c->q[j], c->alpha, &u, &du);
    double fr = orc_weighted_du(W_LONG, r, c->rc, c->h, c->rE, u, du);
    for (int k = 0; k < 3; ++k) F[k] = fr * d[k] / r;
    return fabs(fr);
}
static double fij_lj(const orc_ctx *c, int i, int j, double F[3]) {
    double d[3];
    min_image(c, &c->x[3 * i], &c->x[3 * j], d);
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double u, du;
    orc_u_lj(r, sqrt(c->sig[i] * c->sig[j]), sqrt(c->eps[i] * c->eps[j]), &u, &du);
    double fr = orc_weighted_du(W_LONG, r, c->rc, c->h, c->rE, u, du);
    for (int k = 0; k < 3; ++k) F[k] = fr * d[k] / r;
    return fabs(fr);
}

/* ------------------------------------------------------------------ */
/* bounds L (R-7): sup on a dense grid, times (1 + 1e-6)               */
/* ------------------------------------------------------------------ */
static double sup_coul(const orc_ctx *c, double lo, double hi) {
    if (!(hi > lo)) return 0.0;
    double best = 0.0;
    long K = (long)floor((hi - lo) / 1e-4);
    for (long k = 0; k <= K + 1; ++k) {
        double r = (k <= K) ? lo + 1e-4 * (double)k : hi;
        if (r > hi) r = hi;
        double u, du;
        orc_u_coul(r, ORC_COULOMB, c->alpha, &u, &du);
        double chi, dchi;
        orc_chi(r, c->rc, c->h, &chi, &dchi);
        double g = fabs((1.0 - chi) * du - dchi * u);
        if (g > best) best = g;
    }
    return best * (1.0 + 1e-6);
}
static double sup_lj(const orc_ctx *c, double lo, double hi) { /* 4 eps = 1; sup over sigma range too */
    if (!(hi > lo) || !(c->sig_max > 0.0)) return 0.0;
    double best = 0.0;
    int NS = (c->sig_max > c->sig_min) ? 65 : 1;
    long K = (long)floor((hi - lo) / 1e-4);
    for (int s = 0; s < NS; ++s) {
        double sig = (NS == 1) ? c->sig_min : c->sig_min + (c->sig_max - c->sig_min) * (double)s / (double)(NS - 1);
        for (long k = 0; k <= K + 1; ++k) {
            double r = (k <= K) ? lo + 1e-4 * (double)k : hi;
            if (r > hi) r = hi;
            double u, du;
            orc_u_lj(r, sig, 0.25, &u, &du);
            double chi, dchi;
            orc_chi(r, c->rc, c->h, &chi, &dchi);
            double g = fabs((1.0 - chi) * du - dchi * u);
            if (g > best) best = g;
        }
    }
    return best * (1.0 + 1e-6);
}
static double dmin(double a, double b) { return a < b ? a : b; }
static double dmax(double a, double b) { return a > b ? a : b; }

static void compute_bounds(orc_ctx *c) {
    c->qmax = 0.0; c->eps_max = 0.0; c->sig_min = 1e300; c->sig_max = 0.0;
    for (int i = 0; i < c->n; ++i) {
        c->qmax = dmax(c->qmax, fabs(c->q[i]));
        if (c->eps[i] > 0.0) {
            c->eps_max = dmax(c->eps_max, c->eps[i]);
            c->sig_min = dmin(c->sig_min, c->sig[i]);
            c->sig_max = dmax(c->sig_max, c->sig[i]);
        }
    }
    if (c->eps_max == 0.0) { c->sig_min = 0.0; c->sig_max = 0.0; }
    double lo = c->rc - c->h;
    c->G3 = c->GV2 = c->GV3 = 0.0;
    if (c->policy == 1) { /* R-10c: a ring holds the pairs whose CURRENT distance lies in it */
        const double eA = dmin(dmax(c->rA, lo), c->rE), eM = dmin(dmax(c->rM, eA), c->rE);
        c->GM = sup_coul(c, lo, eA); c->GL = sup_coul(c, eA, eM); c->G3 = sup_coul(c, eM, c->rE);
        /* LJ jumps: the same three rings (the ring technique of P:L422-431 applied to Algorithm 5: beyond the
         * switching zone the long LJ gradient falls off like r^-7) */
        c->GV = sup_lj(c, lo, eA); c->GV2 = sup_lj(c, eA, eM); c->GV3 = sup_lj(c, eM, c->rE);
    } else {              /* R-10: rings by build-time distance, reached up to one skin beyond their edges */
        c->GM = sup_coul(c, lo, dmin(c->rM + c->skin, c->rE));
        c->GL = sup_coul(c, dmax(c->rM - c->skin, lo), c->rE);
        c->GV = sup_lj(c, lo, c->rE);
    }
}

/* GM, GL, GV: rings 1, 2 (Coulomb) and the LJ bound of R-10 / of ring 1; G3, GV2, GV3: R-10c only */
void orc_get_bounds(const orc_ctx *c, double out[12]) {
    out[0] = c->GM; out[1] = c->GL; out[2] = c->GV; out[3] = c->qmax;
    out[4] = c->eps_max; out[5] = c->sig_min; out[6] = c->sig_max; out[7] = c->rM;
    out[8] = c->G3; out[9] = c->GV2; out[10] = c->GV3; out[11] = c->rA;
}

/* ------------------------------------------------------------------ */
/* ring rows (R-10)                                         */
/* ------------------------------------------------------------------ */
/* ---- R-10c: the cell universe of the rings L and V -------------------------------------------------------- */
/* The contract grid has gn cells per edge (cell of an atom = floor(x gn / box), key = (cz ny + cy) nx + cx).  The
 * universe U(h) of a home cell h = (cx, cy, cz) is the set of atoms that sat, at the last list build, in a cell
 * (x, y, z) with cyclic offsets a = |z - cz|, b = |y - cy|, e = |x - cx| such that
 *     a <= R_z,  b <= R_y,  rem = reach^2 - (max(a-1,0) w_z)^2 - (max(b-1,0) w_y)^2 > 0,
 *     e <= min(R_x, floor(sqrt(rem) / w_x) + 1),         reach = r_long + skin, w = box / gn, R = ceil(reach / w):
 * every cell some point of which lies within reach of some point of h (and a few more).  Order: ascending cell
 * key, ascending atom index within a cell.  Any pair closer than r_long now was closer than r_long + skin at the
 * build (no atom moves more than skin/2 between builds), so its partner is in U: a superset to draw from
 * uniformly; entries that carry no force at the moment (too far, too close, excluded, the atom itself)
 * are proposals with rate 0, which thinning allows. */
static int cyc_abs(int v, int c0, int n) {
    int o = ((v - c0) % n + n) % n;
    return o < n - o ? o : n - o;
}
static int uni_xreach(const orc_ctx *c, int a, int b) {
    const double wz = c->p.box[2] / c->gnz, wy = c->p.box[1] / c->gny, wx = c->p.box[0] / c->gnx;
    if (a > c->uR[2] || b > c->uR[1]) return -1;
    const double gz = (a > 1 ? a - 1 : 0) * wz, gy = (b > 1 ? b - 1 : 0) * wy;
    const double rem = c->ureach * c->ureach - gz * gz - gy * gy;
    if (!(rem > 0.0)) return -1;
    int v = (int)floor(sqrt(rem) / wx) + 1;
    return v < c->uR[0] ? v : c->uR[0];
}
/* k >= 0: the k-th atom of U(h) (or -1 if k >= |U(h)|); k < 0: |U(h)| */
static int universe_walk(const orc_ctx *c, int h, int k) {
    const int nx = c->gnx, ny = c->gny, nz = c->gnz;
    const int cx = h % nx, cy = (h / nx) % ny, cz = h / (nx * ny);
    int seen = 0;
    for (int z = 0; z < nz; ++z) {
        const int a = cyc_abs(z, cz, nz);
        if (a > c->uR[2]) continue;
        for (int y = 0; y < ny; ++y) {
            const int b = cyc_abs(y, cy, ny);
            const int xm = uni_xreach(c, a, b);
            if (xm < 0) continue;
            for (int x = 0; x < nx; ++x) {
                if (cyc_abs(x, cx, nx) > xm) continue;
                const int key = (z * ny + y) * nx + x, cnt = c->cell_ptr[key + 1] - c->cell_ptr[key];
                if (k >= 0 && k < seen + cnt) return c->cell_atoms[c->cell_ptr[key] + (k - seen)];
                seen += cnt;
            }
        }
    }
    return k >= 0 ? -1 : seen;
}
static void rebuild_universe(orc_ctx *c) {
    const int n = c->n, ncell = c->gnx * c->gny * c->gnz;
    free(c->cell_ptr); free(c->cell_atoms); free(c->home); free(c->uni_cnt);
    c->cell_ptr = calloc(ncell + 1, sizeof(int));
    c->cell_atoms = malloc(sizeof(int) * n);
    c->home = malloc(sizeof(int) * n);
    c->uni_cnt = malloc(sizeof(int) * ncell);
    for (int i = 0; i < n; ++i) { c->home[i] = contract_key(c, &c->x[3 * i]); c->cell_ptr[c->home[i] + 1]++; }
    for (int k = 0; k < ncell; ++k) c->cell_ptr[k + 1] += c->cell_ptr[k];
    int *fill = malloc(sizeof(int) * ncell);
    memcpy(fill, c->cell_ptr, sizeof(int) * ncell);
    for (int i = 0; i < n; ++i) c->cell_atoms[fill[c->home[i]]++] = i; /* ascending i within a cell */
    free(fill);
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(dynamic, 64)
    for (int h = 0; h < ncell; ++h) c->uni_cnt[h] = (c->cell_ptr[h + 1] > c->cell_ptr[h]) ? universe_walk(c, h, -1) : 0;
}
static int universe_count(const orc_ctx *c, int i) { return c->uni_cnt[c->home[i]]; }

static void rebuild_rows(orc_ctx *c) {
    c->last_build = c->step;
    free(c->ptrM); free(c->idxM); free(c->ptrL); free(c->idxL); free(c->ptrV); free(c->idxV);
    c->ptrL = c->idxL = c->ptrV = c->idxV = NULL;
    double s = c->skin, lo = c->rc - c->h - s;
    if (lo < 0.0) lo = 0.0;
    double em = 1e300;
    if (c->policy == 1) {
        /* R-10c: row A lists every pair that can be in ring A before the next build, row B every pair that can be in
         * ring B (they overlap around r_A); ring C draws from the cell universe.  Mass-weighted skin: the pair (i, j)
         * is listed over [ring - s_ij, ring + s_ij), s_ij = (skin/2)(w_i + w_j), w_i = m_i^-1/2 / mean(m^-1/2): an atom
         * may then move w_i skin/2 before the lists have to be rebuilt -- light atoms move farther in the same time
         * (displacement ~ m^-1/2), so one budget per atom lets a water box go 7 steps where a uniform skin/2 allows 4 */
        neighbor_csr_audit(c, c->x, c->rc - c->h, c->rA, 0.5 * s, 0, 0, &c->ptrM, &c->idxM, &em);   /* row A */
        neighbor_csr_audit(c, c->x, c->rA, c->rM, 0.5 * s, 0, 0, &c->ptrL, &c->idxL, &em);         /* row B */
        rebuild_universe(c);
    } else {
        neighbor_csr_audit(c, c->x, lo, c->rM, 0.0, 0, 0, &c->ptrM, &c->idxM, &em);
        neighbor_csr_audit(c, c->x, dmax(c->rM, lo), c->rE + s, 0.0, 0, 0, &c->ptrL, &c->idxL, &em);
        neighbor_csr_audit(c, c->x, lo, c->rE + s, 0.0, 1, 0, &c->ptrV, &c->idxV, &em);
    }
    {   /* contract-grid cell faces (the row order depends on the cell of every atom, R-10) */
        int nn[3] = {c->gnx, c->gny, c->gnz};
        for (int i = 0; i < c->n; ++i)
            for (int k = 0; k < 3; ++k) {
                double w = c->p.box[k] / nn[k], f = wrap1(c->x[3 * i + k], c->p.box[k]) / w;
                double e = fabs(f - floor(f + 0.5)) * w;
                if (nn[k] > 1 && e < em) em = e;
            }
    }
    if (em < c->st.min_list_margin) { c->st.min_list_margin = em; c->st.min_list_margin_step = c->step; }
    memcpy(c->x_build, c->x, sizeof(double) * 3 * c->n);
    c->st.rebuilds++;
}
static double check_displacement(orc_ctx *c) {
    double mx = 0.0;
    for (int i = 0; i < c->n; ++i) {
        double d[3];
        min_image(c, &c->x[3 * i], &c->x_build[3 * i], d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (c->policy == 1) r /= c->w[i]; /* mass-weighted skin: the budget of atom i is w_i skin / 2 */
        if (r > mx) mx = r;
    }
    if (mx > c->st.max_disp) c->st.max_disp = mx;
    return mx;
}
/* R-10: rows M, L, V.  R-10c: row A, row B, the cell universe of the atom's home cell */
void orc_get_row_counts(const orc_ctx *c, int *nM, int *nL, int *nV) {
    for (int i = 0; i < c->n; ++i) {
        nM[i] = c->ptrM[i + 1] - c->ptrM[i];
        nL[i] = c->ptrL[i + 1] - c->ptrL[i];
        nV[i] = c->policy == 1 ? universe_count(c, i) : c->ptrV[i + 1] - c->ptrV[i];
    }
}
int orc_get_row(const orc_ctx *c, int which, int i, int *out, int cap) {
    if (c->policy == 1 && which == 2) {
        int m = universe_count(c, i);
        for (int k = 0; k < m && k < cap; ++k) out[k] = universe_walk(c, c->home[i], k);
        return m;
    }
    const int *ptr = which == 0 ? c->ptrM : (which == 1 ? c->ptrL : c->ptrV);
    const int *idx = which == 0 ? c->idxM : (which == 1 ? c->idxL : c->idxV);
    int m = ptr[i + 1] - ptr[i];
    for (int k = 0; k < m && k < cap; ++k) out[k] = idx[ptr[i] + k];
    return m;
}

/* ------------------------------------------------------------------ */
/* event log                                                           */
/* ------------------------------------------------------------------ */
static void log_event(orc_ctx *c, const orc_event *e) {
#pragma omp critical(orc_log)
    {
        if (e->margin < c->st.min_margin) { c->st.min_margin = e->margin; c->st.min_margin_step = e->step; }
        if (c->p.flags & ORC_F_EVENT_LOG) {
            if (c->n_ev == c->cap_ev) {
                c->cap_ev = c->cap_ev ? 2 * c->cap_ev : 65536;
                c->ev = realloc(c->ev, sizeof(orc_event) * c->cap_ev);
            }
            c->ev[c->n_ev++] = *e;
        }
    }
}
static int cmp_event(const void *a, const void *b) {
    const orc_event *x = a, *y = b;
    if (x->step != y->step) return x->step < y->step ? -1 : 1;
    if (x->stream != y->stream) return x->stream < y->stream ? -1 : 1;
    if (x->atom != y->atom) return x->atom < y->atom ? -1 : 1;
    return x->iter < y->iter ? -1 : (x->iter > y->iter ? 1 : 0);
}
int64_t orc_get_events(orc_ctx *c, orc_event *buf, int64_t cap) {
    qsort(c->ev, c->n_ev, sizeof(orc_event), cmp_event);
    int64_t m = c->n_ev < cap ? c->n_ev : cap;
    if (buf) memcpy(buf, c->ev, sizeof(orc_event) * m);
    return c->n_ev;
}
void orc_clear_events(orc_ctx *c) { c->n_ev = 0; }
void orc_get_stats(const orc_ctx *c, orc_stats *out) { *out = c->st; }
void orc_reset_stats(orc_ctx *c) {
    memset(&c->st, 0, sizeof c->st);
    c->st.min_margin = 1e300;
    c->st.min_list_margin = 1e300;
}

/* ------------------------------------------------------------------ */
/* Jump chains: Algorithm 4 with the ring technique (step C', R-11;    */
/* P:L352-420) and Algorithm 5 (step J', BPS on the long   */
/* LJ part, R-14).  Position x frozen; one chain per atom. */
/* ------------------------------------------------------------------ */
/* One ring of one atom: a set one can draw from uniformly, its size and the bound on |F_ij| over it. */
typedef struct {
    int kind;        /* where the candidates come from: 0 row M, 1 row L, 2 row V, 3 the cell universe (R-10c) */
    int n;           /* number of candidates, N_Y(i) */
    double L;        /* L_{Y,i} */
    double rlo, rhi; /* R-10c: the pair carries its force through this ring while rlo <= r < rhi (current distance);
                        rlo < 0 (R-10): ring membership is list membership */
} orc_ring;

/* the rings of atom i for the Coulomb (lj = 0), the LJ (lj = 1) or the combined (lj = 2, R-22) jumps; returns their number */
static int rings_of(const orc_ctx *c, int i, int lj, orc_ring R[3]) {
    const double cq = fabs(c->q[i]) * c->qmax, ce = 4.0 * sqrt(c->eps[i] * c->eps_max); /* uniform in j: P:L346, L369, L455 */
    const int nA = c->ptrM[i + 1] - c->ptrM[i];
    if (c->policy == 1) { /* R-10c: A = [r_c - h, r_A), B = [r_A, r_M) from the rows, L = [r_M, r_long) from the universe */
        const int nB = c->ptrL[i + 1] - c->ptrL[i], nU = universe_count(c, i);
        /* lj = 2 (R-22): the pair gradient is the sum of the two long parts, bounded by the sum of their bounds */
        const double fq = lj == 1 ? 0.0 : cq, fe = lj == 0 ? 0.0 : ce;
        R[0] = (orc_ring){0, nA, fq * c->GM + fe * c->GV, c->rc - c->h, c->rA};
        R[1] = (orc_ring){1, nB, fq * c->GL + fe * c->GV2, c->rA, c->rM};
        R[2] = (orc_ring){3, nU, fq * c->G3 + fe * c->GV3, c->rM, c->rE};
        return 3;
    }
    if (lj) { R[0] = (orc_ring){2, c->ptrV[i + 1] - c->ptrV[i], ce * c->GV, -1.0, 0.0}; return 1; }
    R[0] = (orc_ring){0, nA, cq * c->GM, -1.0, 0.0};
    R[1] = (orc_ring){1, c->ptrL[i + 1] - c->ptrL[i], cq * c->GL, -1.0, 0.0};
    return 2;
}
static int ring_candidate(const orc_ctx *c, int i, const orc_ring *R, int k) {
    switch (R->kind) {
        case 0: return c->idxM[c->ptrM[i] + k];
        case 1: return c->idxL[c->ptrL[i] + k];
        case 2: return c->idxV[c->ptrV[i] + k];
        default: return universe_walk(c, c->home[i], k);
    }
}

/* F_ij of the mechanism run by chain_atom: lj = 0 the long Coulomb gradient, 1 the long LJ gradient, 2 their sum (R-22) */
static double fij_mode(const orc_ctx *c, int lj, int i, int j, double F[3]) {
    if (lj == 0) return fij_coul(c, i, j, F);
    if (lj == 1) return fij_lj(c, i, j, F);
    double Fl[3];
    fij_coul(c, i, j, F);
    fij_lj(c, i, j, Fl);
    for (int k = 0; k < 3; ++k) F[k] += Fl[k];
    return sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
}

/* lj = 2 (R-22, ORC_F_COMBINED): as lj = 0 with F_ij the whole long pair gradient and L_Y the sum of the two bounds.
 * lj = 0: step (C') for atom i, general mechanism (6),(7) with eps (or BPS, eps = inf), acceleration a between
 * proposals.  lj = 1: step (J'), BPS (4),(5) on the long LJ part, a = 0 (the caller passes zeros): the same loop
 * with the constant bound beta |v| sum N_Y L_Y (|v| is preserved by reflections), so that the number of
 * proposals is Poisson as Algorithm 5 asks (R-14).
 * Draws of a proposal, from one Philox block (R-15): E, ring, k, U; G~ attempts draw from stream + 16. */
static void chain_atom(orc_ctx *c, int i, int lj, double H, const double a[3], int stream, int64_t step,
                       int64_t *n_prop, int64_t *n_acc, int64_t *n_gt, int64_t *n_exp, double *max_p, double *max_gl) {
    if (lj == 1 && !(c->eps[i] > 0.0)) return; /* no LJ on this atom: no chain */
    double *v = &c->v[3 * i];
    const double eps = lj == 1 ? INFINITY : c->p.eps_jump, sbm = c->sbm[i], beta = c->beta;
    const int bps = isinf(eps);
    /* R-19 (NEXT-1): eps_mode 1 = adaptive eps(x) = eps0 |F_ij(x)|, eps0 = eps_jump.  With
     * g = |F_ij| <= L_Y, eta = eps0 g sqrt(beta m)(v.n) and Theta(eta) <= eta_+ + 1/sqrt(2 pi) the pair rate
     * lambda_ij = sqrt(beta) Theta(eta) / (eps0 sqrt(m)) (P:L340 with eps = eps0 g) is bounded, uniformly in j, by
     * lambda*_Y = beta L_Y B_v + (1/eps0) sqrt(beta / (2 pi m)); p = lambda_ij / lambda*_Y. */
    const int adaptive = c->p.eps_mode == 1 && !bps;
    orc_ring R[3];
    const int nr = rings_of(c, i, lj, R);
    double S = 0.0; /* sum_Y N_Y L_Y */
    int ntot = 0;
    for (int y = 0; y < nr; ++y) { S += (double)R[y].n * R[y].L; ntot += R[y].n; }
    if (lj == 1 && !(S > 0.0)) return; /* (J') without a partner: nothing to log, as under Algorithm 5 with N = 0 */
    double t = 0.0;
    uint32_t block = 0;  /* proposal k of the chain draws Philox block k of its stream ...                     */
    uint32_t gblock = 0; /* ... and the G~ attempts draw blocks 0, 1, ... of stream + 16 (R-15)                 */
    uint32_t w[4];
    /* R-11: Algorithm 4 prints B_v and lambda-bar inside the loop, i.e. re-evaluated at every proposal;
     * P:L161 says local bounds "need to be re-evaluated after each jump".  B_v bounds |v_i| on the whole of
     * [t, delta/2] and between two accepted jumps v_i only drifts with a_i, so the bound evaluated at t = 0
     * or after an ACCEPTED jump stays valid until the next accepted jump: by default (bound_every = 0) it is held in
     * between ("epoch" form: looser, hence a few more proposals, the same law by P:L157); bound_every = 1 is the
     * literal per-proposal form (orc_set_bound_mode; tests/test_oracle_pins.py compares the two). */
    int fresh = 1;
    double Bv = 0.0, lam = 0.0;
    double wgt[3] = {0.0, 0.0, 0.0}; /* ring Y is picked with probability wgt[Y] / sum wgt */
    const double lam0 = bps ? 0.0 : (1.0 / eps) * beta * ORC_INV_SQRT_2PI / sbm; /* (1/eps) sqrt(beta/(2 pi m)) */
    const double a2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
    for (int iter = 0;; ++iter) {
        orc_event ev;
        memset(&ev, 0, sizeof ev);
        ev.step = (int32_t)step; ev.stream = stream; ev.atom = i; ev.iter = iter; ev.ring = -1; ev.j = -1;
        double mg = 1e300;
        double tau = H - t;
        if (fresh || c->bound_every) {
            double va = v[0] * a[0] + v[1] * a[1] + v[2] * a[2];
            double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
            Bv = sqrt(v2 + tau * tau * a2 + 2.0 * tau * (va > 0.0 ? va : 0.0));
            lam = 0.0;
            for (int y = 0; y < nr; ++y) {
                if (!(S > 0.0)) wgt[y] = 0.0; /* no partner, or an uncharged atom: no mechanism */
                else if (adaptive) wgt[y] = (double)R[y].n * (beta * R[y].L * Bv + lam0); /* sum of lambda*_Y (R-19) */
                else wgt[y] = (double)R[y].n * R[y].L;
                lam += wgt[y];
            }
            if (!adaptive) lam *= beta * Bv + lam0; /* P:L374; (J'): beta |v| sum N_Y L_Y */
            fresh = 0;
        }
        chain_block(c, i, step, stream, block++, w);
        double E = -log(orc_u01(w[0]));
        double T = lam > 0.0 ? E / lam : INFINITY;
        ev.T = T;
        if (isfinite(T)) mg = upd(mg, (t + T - H) / H);
        if (t + T > H) {
            v[0] += tau * a[0]; v[1] += tau * a[1]; v[2] += tau * a[2];
            ev.margin = mg;
            (*n_exp)++;
            log_event(c, &ev);
            break;
        }
        t += T;
        v[0] += T * a[0]; v[1] += T * a[1]; v[2] += T * a[2];
        /* ring pick: the first ring whose cumulated weight exceeds ur * (sum of weights) */
        double ur = orc_u01(w[1]), wsum = 0.0, cum = 0.0;
        for (int y = 0; y < nr; ++y) wsum += wgt[y];
        int ring = 0;
        for (int y = 0; y < nr; ++y) {
            cum += wgt[y];
            ring = y;
            if (y < nr - 1 && wgt[y] > 0.0) mg = upd(mg, ur - cum / wsum);
            if (ur * wsum < cum) break;
        }
        while (R[ring].n == 0 && ring > 0) --ring; /* (rounding at the upper end: fall back to a ring that has entries) */
        while (R[ring].n == 0 && ring < nr - 1) ++ring;
        int k = (int)(((uint64_t)w[2] * (uint64_t)R[ring].n) >> 32);
        int j = ring_candidate(c, i, &R[ring], k);
        double LY = R[ring].L;
        double U = orc_u01(w[3]);
        ev.ring = 4 * lj + ring; ev.j = j; ev.U = U; /* ring codes 0-2 (C'), 4-6 (J'), 8-10 (combined) */
        (*n_prop)++;
        double F[3];
        double g = 0.0;
        if (R[ring].rlo < 0.0) g = fij_mode(c, lj, i, j, F); /* R-10 */
        else if (j != i && !(R[ring].kind == 3 && is_excluded(c, i, j))) {
            /* R-10c: the pair carries its force through the ring its CURRENT distance lies in; drawn
             * through another ring it has rate 0 -- every pair is counted exactly once.  The universe also holds
             * the atom itself and its excluded partners: rate 0 (the rows never list them, R-9). */
            double d[3];
            min_image(c, &c->x[3 * i], &c->x[3 * j], d);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            mg = upd(mg, r - R[ring].rlo);
            mg = upd(mg, r - R[ring].rhi);
            if (r >= R[ring].rlo && r < R[ring].rhi) g = fij_mode(c, lj, i, j, F);
        }
        if (g > 0.0) {
            if (g / LY > *max_gl) *max_gl = g / LY;
            double n[3] = {F[0] / g, F[1] / g, F[2] / g};
            double vn = v[0] * n[0] + v[1] * n[1] + v[2] * n[2];
            double p;
            const double eps_ij = adaptive ? eps * g : eps; /* eps(x) = eps0 |F_ij(x)| */
            if (bps) p = (vn > 0.0 ? vn : 0.0) * g / (LY * Bv); /* (4) over the bound; (J'): P:L486 with B_v = |v| */
            else if (adaptive) p = orc_theta(eps_ij * sbm * vn) / (eps * sbm * LY * Bv + ORC_INV_SQRT_2PI); /* R-19 */
            else p = g * orc_theta(eps * sbm * vn) / (LY * (Bv * eps * sbm + ORC_INV_SQRT_2PI)); /* P:L397 + sqrt(beta) */
            ev.p = p;
            if (p > *max_p) *max_p = p;
            mg = upd(mg, U - p);
            if (U <= p) {
                double gt = 0.0;
                int att = 0;
                if (!bps) gt = orc_gtilde(c, eps_ij * sbm * vn, i, step, stream + 16, &gblock, &att, &mg);
                orc_jump_kick(eps_ij, sbm, n, gt, v); /* P:L406; eps = inf: reflection (5) */
                ev.accepted = 1; ev.gt = gt; ev.n_gt = att;
                (*n_acc)++;
                (*n_gt) += att;
                fresh = 1;
            }
        }
        ev.margin = mg;
        log_event(c, &ev);
    }
    (void)ntot;
}

/* C over all atoms; acc_src: gradient array giving a = -M^-1 F (NULL -> a = 0) */
static void phase_C(orc_ctx *c, double H, const double *grad, int stream, int64_t step, int mode) {
    int64_t np = 0, nacc = 0, ngt = 0, nexp = 0;
    double mp = 0.0, mgl = 0.0;
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(dynamic, 64) reduction(+ : np, nacc, ngt, nexp) reduction(max : mp, mgl)
    for (int i = 0; i < c->n; ++i) {
        double a[3] = {0, 0, 0};
        if (grad)
            for (int k = 0; k < 3; ++k) a[k] = -(ORC_KCAL / c->m[i]) * grad[3 * i + k];
        chain_atom(c, i, mode, H, a, stream, step, &np, &nacc, &ngt, &nexp, &mp, &mgl);
    }
    c->st.proposals += np; c->st.accepts += nacc; c->st.gt_attempts += ngt; c->st.expiries += nexp;
    if (mp > c->st.max_p) c->st.max_p = mp;
    if (mgl > c->st.max_g_over_L) c->st.max_g_over_L = mgl;
}
static void phase_J(orc_ctx *c, double H, int stream, int64_t step) {
    int64_t np = 0, nacc = 0, ngt = 0, nexp = 0;
    double mp = 0.0, mgl = 0.0;
    const double zero[3] = {0.0, 0.0, 0.0};
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(dynamic, 64) reduction(+ : np, nacc, ngt, nexp) reduction(max : mp, mgl)
    for (int i = 0; i < c->n; ++i) chain_atom(c, i, 1, H, zero, stream, step, &np, &nacc, &ngt, &nexp, &mp, &mgl);
    c->st.proposals += np; c->st.accepts += nacc; c->st.expiries += nexp;
    if (mp > c->st.max_p) c->st.max_p = mp;
    if (mgl > c->st.max_g_over_L) c->st.max_g_over_L = mgl;
}
/* plain (B): v <- v - H M^-1 F, written as v += H a so that it is bit-identical to an event-free (C) */
static void phase_B(orc_ctx *c, double H, const double *grad) {
    for (int i = 0; i < c->n; ++i)
        for (int k = 0; k < 3; ++k) {
            double a = -(ORC_KCAL / c->m[i]) * grad[3 * i + k];
            c->v[3 * i + k] += H * a;
        }
}
/* C' then J' (fwd) or J' then C' (reverse) over a duration H */
static void jump_phase(orc_ctx *c, double H, const double *grad, int sC, int sJ, int64_t step, int reverse) {
    int coul = (c->p.flags & ORC_F_COUL_JUMPS) != 0, lj = (c->p.flags & ORC_F_LJ_JUMPS) != 0;
    if (c->p.flags & ORC_F_COMBINED) { /* R-22: one mechanism for the whole long pair gradient, no (J') */
        phase_C(c, H, grad, sC, step, 2);
        return;
    }
    if (reverse && lj) phase_J(c, H, sJ, step);
    if (coul) phase_C(c, H, grad, sC, step, 0);
    else if (grad) phase_B(c, H, grad);
    if (!reverse && lj) phase_J(c, H, sJ, step);
}

/* (A) P:L119 and (O) P:L121-123 */
static void phase_A(orc_ctx *c, double H) {
    for (int k = 0; k < 3 * c->n; ++k) { c->x[k] += H * c->v[k]; c->xu[k] += H * c->v[k]; }
}
static void phase_O(orc_ctx *c, double dt, int64_t step) {
    double c1 = exp(-c->p.gamma_per_ps * dt), c2 = sqrt(1.0 - c1 * c1);
    for (int i = 0; i < c->n; ++i) {
        uint32_t w[4];
        chain_block(c, i, step, 0, 0, w);
        double r1 = sqrt(-2.0 * log(orc_u01(w[0]))), a1 = 2.0 * ORC_PI * orc_u01(w[1]);
        double r2 = sqrt(-2.0 * log(orc_u01(w[2]))), a2 = 2.0 * ORC_PI * orc_u01(w[3]);
        double G[3] = {r1 * cos(a1), r1 * sin(a1), r2 * cos(a2)};
        for (int k = 0; k < 3; ++k) c->v[3 * i + k] = c1 * c->v[3 * i + k] + c2 / c->sbm[i] * G[k];
    }
}
static void wrap_all(orc_ctx *c) {
    for (int i = 0; i < c->n; ++i)
        for (int k = 0; k < 3; ++k) c->x[3 * i + k] = wrap1(c->x[3 * i + k], c->p.box[k]);
}
/* A O A, wrap, step counter, scheduled rebuild (steps 3-6 of C.3) */
static void aoa_and_lists(orc_ctx *c) {
    phase_A(c, 0.5 * c->dt);
    phase_O(c, c->dt, c->step);
    phase_A(c, 0.5 * c->dt);
    wrap_all(c);
    c->step++;
    const double mx = check_displacement(c);
    /* R-10c list schedule, counted from the LAST build: P = nlist_every steps after it at the latest, and -- from
     * Q = min(3, P/4) steps after it on -- as soon as some atom has used up its share of the skin, w_i skin/2 (the lists are supersets
     * of what they must hold while no atom has; water, skin 1 A: 6 to 9 steps).  The test on the displacement is
     * one more discontinuous decision (R-17): its margin is audited with those of the lists.  (Round-1 policy 0:
     * every P-th step, nothing else.) */
    const int P = c->p.nlist_every;
    const long long age = c->step - c->last_build;
    int rebuild = P > 0 && (c->policy == 1 ? age >= P : c->step % P == 0);
    if (!rebuild && c->policy == 1 && P > 0 && age >= (P >= 12 ? 3 : (P >= 4 ? P / 4 : 1))) {
        const double e = fabs(mx - 0.5 * c->skin);
        if (e < c->st.min_list_margin) { c->st.min_list_margin = e; c->st.min_list_margin_step = c->step; }
        rebuild = mx > 0.5 * c->skin;
    }
    if (rebuild) rebuild_rows(c);
}

/* ------------------------------------------------------------------ */
/* Reciprocal part of the Ewald sum ("Ewald summation"; the paper's SPME is an FFT approximation of exactly */
/* this sum and is out of scope: here the sum itself, as the slow many-body force F_{0,1} of P:L137-145, R-21).   */
/*   U_rec  = (C / 2V) sum_{k != 0} (4 pi / k^2) exp(-k^2 / 4 alpha^2) |S(k)|^2,  S(k) = sum_j q_j exp(i k.x_j),   */
/*            k = 2 pi (nx/Lx, ny/Ly, nz/Lz), all |k| <= k_cut; k and -k give the same term: sum over a half space. */
/*   U_self = -C alpha / sqrt(pi) sum_i q_i^2 (constant)                                                           */
/*   U_excl = -sum_{excluded pairs i<j} C q_i q_j erf(alpha r_ij) / r_ij: the reciprocal sum contains every pair,   */
/*            also those that R-9 excludes from the direct sum; their smooth part is taken out again.               */
/* ------------------------------------------------------------------ */
void orc_ewald_setup(orc_ctx *c, double k_cut) {
    free(c->kn); c->kn = NULL; c->nk = 0;
    if (!(c->alpha > 0.0)) return;
    if (!(k_cut > 0.0)) k_cut = 8.0 * c->alpha; /* exp(-k^2/4 alpha^2) = e^-16 = 1.1e-7, the size of erfc(3.8) (R-2) */
    int nmax[3];
    for (int d = 0; d < 3; ++d) nmax[d] = (int)floor(k_cut * c->p.box[d] / (2.0 * ORC_PI));
    for (int pass = 0; pass < 2; ++pass) {
        int cnt = 0;
        for (int nx = 0; nx <= nmax[0]; ++nx)
            for (int ny = (nx == 0 ? 0 : -nmax[1]); ny <= nmax[1]; ++ny)
                for (int nz = ((nx == 0 && ny == 0) ? 1 : -nmax[2]); nz <= nmax[2]; ++nz) {
                    double kx = 2.0 * ORC_PI * nx / c->p.box[0], ky = 2.0 * ORC_PI * ny / c->p.box[1], kz = 2.0 * ORC_PI * nz / c->p.box[2];
                    if (kx * kx + ky * ky + kz * kz > k_cut * k_cut) continue;
                    if (pass) { c->kn[3 * cnt] = nx; c->kn[3 * cnt + 1] = ny; c->kn[3 * cnt + 2] = nz; }
                    ++cnt;
                }
        if (!pass) { c->nk = cnt; c->kn = malloc(sizeof(int) * 3 * (cnt > 0 ? cnt : 1)); }
    }
}
int orc_ewald_nk(const orc_ctx *c) { return c->nk; }
/* adds grad (U_rec + U_excl) to out (kcal/mol/A), returns U_rec + U_self + U_excl (kcal/mol) */
static double slow_accumulate(const orc_ctx *c, double *out) {
    const int n = c->n, nk = c->nk;
    const double V = c->p.box[0] * c->p.box[1] * c->p.box[2];
    double e = 0.0;
    double *Sr = malloc(sizeof(double) * (nk > 0 ? nk : 1)), *Si = malloc(sizeof(double) * (nk > 0 ? nk : 1));
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(static)
    for (int m = 0; m < nk; ++m) {
        const double kx = 2.0 * ORC_PI * c->kn[3 * m] / c->p.box[0], ky = 2.0 * ORC_PI * c->kn[3 * m + 1] / c->p.box[1],
                     kz = 2.0 * ORC_PI * c->kn[3 * m + 2] / c->p.box[2];
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            const double th = kx * c->x[3 * j] + ky * c->x[3 * j + 1] + kz * c->x[3 * j + 2];
            sr += c->q[j] * cos(th); si += c->q[j] * sin(th);
        }
        Sr[m] = sr; Si[m] = si;
    }
    for (int m = 0; m < nk; ++m) {
        const double kx = 2.0 * ORC_PI * c->kn[3 * m] / c->p.box[0], ky = 2.0 * ORC_PI * c->kn[3 * m + 1] / c->p.box[1],
                     kz = 2.0 * ORC_PI * c->kn[3 * m + 2] / c->p.box[2];
        const double k2 = kx * kx + ky * ky + kz * kz;
        /* half space: twice the (1/2V) term */
        e += (ORC_COULOMB / V) * (4.0 * ORC_PI / k2) * exp(-k2 / (4.0 * c->alpha * c->alpha)) * (Sr[m] * Sr[m] + Si[m] * Si[m]);
    }
#pragma omp parallel for num_threads(orc_threads(c->n)) schedule(static)
    for (int i = 0; i < n; ++i) {
        double g[3] = {0, 0, 0};
        for (int m = 0; m < nk; ++m) {
            const double kx = 2.0 * ORC_PI * c->kn[3 * m] / c->p.box[0], ky = 2.0 * ORC_PI * c->kn[3 * m + 1] / c->p.box[1],
                         kz = 2.0 * ORC_PI * c->kn[3 * m + 2] / c->p.box[2];
            const double k2 = kx * kx + ky * ky + kz * kz;
            const double A = (ORC_COULOMB / V) * (4.0 * ORC_PI / k2) * exp(-k2 / (4.0 * c->alpha * c->alpha));
            const double th = kx * c->x[3 * i] + ky * c->x[3 * i + 1] + kz * c->x[3 * i + 2];
            /* d|S|^2/dx_i = 2 q_i k (S_i cos th - S_r sin th) */
            const double t = 2.0 * A * c->q[i] * (Si[m] * cos(th) - Sr[m] * sin(th));
            g[0] += t * kx; g[1] += t * ky; g[2] += t * kz;
        }
        for (int d = 0; d < 3; ++d) out[3 * i + d] += g[d];
    }
    free(Sr); free(Si);
    if (nk > 0) {
        for (int i = 0; i < n; ++i) e -= ORC_COULOMB * c->alpha / sqrt(ORC_PI) * c->q[i] * c->q[i];
        if (c->excl_ptr)
            for (int i = 0; i < n; ++i)
                for (int t = c->excl_ptr[i]; t < c->excl_ptr[i + 1]; ++t) {
                    const int j = c->excl_idx[t];
                    if (j <= i) continue;
                    double d[3];
                    min_image(c, &c->x[3 * i], &c->x[3 * j], d);
                    const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]), qq = ORC_COULOMB * c->q[i] * c->q[j];
                    const double ar = c->alpha * r;
                    e -= qq * erf(ar) / r;
                    /* d/dr [-qq erf(alpha r)/r] = -qq [ (2 alpha/sqrt pi) exp(-alpha^2 r^2) / r - erf(alpha r) / r^2 ] */
                    const double du = -qq * (2.0 * c->alpha / sqrt(ORC_PI) * exp(-ar * ar) / r - erf(ar) / (r * r));
                    for (int k = 0; k < 3; ++k) { out[3 * i + k] += du * d[k] / r; out[3 * j + k] -= du * d[k] / r; }
                }
    }
    return e;
}
static void compute_slow(orc_ctx *c) {
    memset(c->f_slow, 0, sizeof(double) * 3 * c->n);
    slow_accumulate(c, c->f_slow);
}

/* ------------------------------------------------------------------ */
/* public steps                                                        */
/* ------------------------------------------------------------------ */
/* C'J'AOAJ'C' */
void orc_jump_step(orc_ctx *c, int nsteps) {
    const double H = 0.5 * c->dt;
    for (int s = 0; s < nsteps; ++s) {
        int64_t st = c->step;
        if (c->p.flags & ORC_F_BJAOAJB) {
            /* B J A O A J B (NEXT-3): the kick by F0 apart from the jumps, which run on a piecewise
             * constant velocity (W of P:L125) -- within (J) the Coulomb chains then the LJ chains, mirrored. */
            phase_B(c, H, c->f0);
            jump_phase(c, H, NULL, 1, 2, st, 0);
            aoa_and_lists(c);
            compute_f0(c);
            jump_phase(c, H, NULL, 4, 3, st, 1);
            phase_B(c, H, c->f0);
            continue;
        }
        jump_phase(c, H, c->f0, 1, 2, st, 0);
        aoa_and_lists(c);
        compute_f0(c);
        jump_phase(c, H, c->f0, 4, 3, st, 1);
    }
}
/* BAOAB with the unsplit force to r_long (P:L112-125 without J) */
void orc_baoab_step(orc_ctx *c, int nsteps) {
    double *f = malloc(sizeof(double) * 3 * c->n);
    compute_full(c, f);
    for (int s = 0; s < nsteps; ++s) {
        phase_B(c, 0.5 * c->dt, f);
        aoa_and_lists(c);
        compute_full(c, f);
        phase_B(c, 0.5 * c->dt, f);
    }
    free(f);
    compute_f0(c);
}
/* JUMP-RESPA / BAOAB-RESPA (R-12).  long_in_outer: the comparator's kick carries the long pair gradient
 * (two-level BAOAB-RESPA); 0 when a third level carries it (BAOAB-RESPA1). */
static void respa_outer_steps(orc_ctx *c, int nouter, int long_in_outer) {
    const int n = c->p.n_inner;
    const double D = n * c->dt;
    const int paper = (c->p.flags & ORC_F_RESPA_PAPER) != 0, cmp = (c->p.flags & ORC_F_RESPA_COMPARATOR) != 0;
    double *fout = malloc(sizeof(double) * 3 * c->n);
    for (int o = 0; o < nouter; ++o) {
        for (int half = 0; half < 2; ++half) {
            if (half == 1) { /* inner loop: n x BAOAB_delta with F_in */
                for (int s = 0; s < n; ++s) {
                    const double *fin = paper ? c->f_bond : c->f0;
                    phase_B(c, 0.5 * c->dt, fin);
                    aoa_and_lists(c);
                    if (paper) compute_bonded_only(c); else compute_f0(c);
                    phase_B(c, 0.5 * c->dt, paper ? c->f_bond : c->f0);
                }
                if (paper) compute_f0(c); /* short non-bonded at the new x for the closing outer phase */
            }
            if (cmp) {
                if (long_in_outer) compute_long(c);
                for (int k = 0; k < 3 * c->n; ++k) fout[k] = (long_in_outer ? c->f_long[k] : 0.0) + (paper ? c->f_nb[k] : 0.0);
                phase_B(c, 0.5 * D, fout);
            } else {
                const double *grad = paper ? c->f_nb : NULL;
                if (half == 0) jump_phase(c, 0.5 * D, grad, 5, 6, c->outer, 0);
                else jump_phase(c, 0.5 * D, grad, 8, 7, c->outer, 1);
            }
        }
        c->outer++;
    }
    free(fout);
}
void orc_jump_respa_step(orc_ctx *c, int nouter) { respa_outer_steps(c, nouter, 1); }

/* JUMP-RESPA1 / BAOAB-RESPA1 ("can itself be iterated"; R-21): three levels delta, kappa = m delta
 * (m = n_inner), Delta = n_mid kappa.  delta: intramolecular; kappa: short-range non-bonded and the jumps -- the
 * "paper" placement of the two-level driver above; Delta: the slow many-body force F_{0,1} = grad(U_rec + U_excl),
 *   v <- v - (Delta/2) M^-1 F_{0,1}(x);  n_mid x [middle step of size kappa];  v <- v - (Delta/2) M^-1 F_{0,1}(x).
 * Comparator (ORC_F_RESPA_COMPARATOR): the long pair gradient rides with F_{0,1} in the outermost kick
 * and the middle level kicks with the short non-bonded gradient only. */
void orc_jump_respa1_step(orc_ctx *c, int nouter, int n_mid) {
    const int cmp = (c->p.flags & ORC_F_RESPA_COMPARATOR) != 0;
    const uint32_t keep = c->p.flags;
    const double D = (double)n_mid * c->p.n_inner * c->dt;
    if (!c->f_slow) c->f_slow = calloc(3 * c->n, sizeof(double));
    double *fo = malloc(sizeof(double) * 3 * c->n);
    c->p.flags |= ORC_F_RESPA_PAPER;
    for (int o = 0; o < nouter; ++o) {
        for (int half = 0; half < 2; ++half) {
            if (half == 1) respa_outer_steps(c, n_mid, 0);
            compute_slow(c);
            if (cmp) compute_long(c);
            for (int k = 0; k < 3 * c->n; ++k) fo[k] = c->f_slow[k] + (cmp ? c->f_long[k] : 0.0);
            phase_B(c, 0.5 * D, fo);
        }
        c->outer1++;
    }
    c->p.flags = keep;
    free(fo);
}

/* ------------------------------------------------------------------ */
/* life cycle                                                          */
/* ------------------------------------------------------------------ */
static void *dup_mem(const void *src, size_t bytes) {
    void *p = malloc(bytes > 0 ? bytes : 1);
    if (src && bytes) memcpy(p, src, bytes);
    return p;
}
orc_ctx *orc_create(const orc_params *p, const double *pos, const double *vel, const double *mass,
                    const double *charge, const double *sigma, const double *eps, int n_bonds, const int *bond_ij,
                    const double *bond_k, const double *bond_r0, int n_angles, const int *angle_ijk,
                    const double *angle_k, const double *angle_t0, const int *excl_ptr, const int *excl_idx) {
    orc_ctx *c = calloc(1, sizeof(orc_ctx));
    c->p = *p;
    int n = c->n = p->n_atoms;
    c->x = dup_mem(pos, sizeof(double) * 3 * n);
    c->xu = dup_mem(pos, sizeof(double) * 3 * n);
    c->v = dup_mem(vel, sizeof(double) * 3 * n);
    c->m = dup_mem(mass, sizeof(double) * n);
    c->q = dup_mem(charge, sizeof(double) * n);
    c->sig = dup_mem(sigma, sizeof(double) * n);
    c->eps = dup_mem(eps, sizeof(double) * n);
    c->nb = n_bonds; c->na = n_angles;
    c->bij = dup_mem(bond_ij, sizeof(int) * 2 * n_bonds);
    c->bk = dup_mem(bond_k, sizeof(double) * n_bonds);
    c->br0 = dup_mem(bond_r0, sizeof(double) * n_bonds);
    c->aijk = dup_mem(angle_ijk, sizeof(int) * 3 * n_angles);
    c->ak = dup_mem(angle_k, sizeof(double) * n_angles);
    c->at0 = dup_mem(angle_t0, sizeof(double) * n_angles);
    if (excl_ptr) {
        c->excl_ptr = dup_mem(excl_ptr, sizeof(int) * (n + 1));
        c->excl_idx = dup_mem(excl_idx, sizeof(int) * excl_ptr[n]);
    }
    c->kT = ORC_KB * p->temperature_K;
    c->beta = 1.0 / c->kT;
    c->dt = p->dt_fs * 1e-3;
    c->rc = p->r_short; c->h = p->r_switch; c->rE = p->r_long; c->skin = p->skin;
    c->alpha = p->ewald_alpha < 0.0 ? 3.8 / p->r_long : p->ewald_alpha; /* R-2 */
    /* r_mid <= 0: no ring, M is empty and L covers the whole shell */
    c->rA = p->r_mid_in > 0.0 ? p->r_mid_in : c->rc; /* R-10c: ring A = the switching zone by default */
    if (p->r_mid > 0.0) c->rM = p->r_mid;
    else c->rM = p->list_policy == 1 ? c->rA : dmax(c->rc - c->h - c->skin, 0.0); /* no split asked for */
    if (c->rA > c->rM) c->rA = c->rM;
    c->sbm = malloc(sizeof(double) * n);
    for (int i = 0; i < n; ++i) c->sbm[i] = sqrt(c->m[i] / (c->kT * ORC_KCAL));
    c->w = malloc(sizeof(double) * n);
    {
        double sum = 0.0;
        for (int i = 0; i < n; ++i) sum += 1.0 / sqrt(c->m[i]);
        c->w_max = 0.0;
        for (int i = 0; i < n; ++i) {
            c->w[i] = p->list_policy == 1 ? (1.0 / sqrt(c->m[i])) / (sum / n) : 1.0;
            if (c->w[i] > c->w_max) c->w_max = c->w[i];
        }
    }
    double edge = p->cell_edge > 0.0 ? p->cell_edge : (p->r_long + p->skin * c->w_max) / 4.0;
    c->gnx = (int)floor(p->box[0] / edge); if (c->gnx < 1) c->gnx = 1;
    c->gny = (int)floor(p->box[1] / edge); if (c->gny < 1) c->gny = 1;
    c->gnz = (int)floor(p->box[2] / edge); if (c->gnz < 1) c->gnz = 1;
    c->policy = p->list_policy == 1 ? 1 : 0;
    c->ureach = p->r_long + p->skin * c->w_max;
    {
        int nn[3] = {c->gnx, c->gny, c->gnz};
        for (int k = 0; k < 3; ++k) c->uR[k] = (int)ceil(c->ureach / (p->box[k] / nn[k]));
    }
    c->x_build = malloc(sizeof(double) * 3 * n);
    c->f_bond = calloc(3 * n, sizeof(double));
    c->f_nb = calloc(3 * n, sizeof(double));
    c->f0 = calloc(3 * n, sizeof(double));
    c->f_long = calloc(3 * n, sizeof(double));
    orc_reset_stats(c);
    wrap_all(c);
    compute_bounds(c);
    rebuild_rows(c);
    compute_f0(c);
    return c;
}
void orc_free(orc_ctx *c) {
    if (!c) return;
    free(c->x); free(c->xu); free(c->v); free(c->m); free(c->q); free(c->sig); free(c->eps);
    free(c->bij); free(c->bk); free(c->br0); free(c->aijk); free(c->ak); free(c->at0);
    free(c->excl_ptr); free(c->excl_idx); free(c->sbm); free(c->x_build);
    free(c->ptrM); free(c->idxM); free(c->ptrL); free(c->idxL); free(c->ptrV); free(c->idxV);
    free(c->f_bond); free(c->f_nb); free(c->f0); free(c->f_long); free(c->ev); free(c->kn); free(c->f_slow);
    free(c->cell_ptr); free(c->cell_atoms); free(c->home); free(c->uni_cnt); free(c->w);
    free(c);
}
/* which: 0 wrapped x, 1 v, 2 unwrapped x */
void orc_get_state(const orc_ctx *c, int which, double *out) {
    const double *src = which == 0 ? c->x : (which == 1 ? c->v : c->xu);
    memcpy(out, src, sizeof(double) * 3 * c->n);
}
/* overwrite x (and v); rows and F0 are refreshed */
void orc_set_state(orc_ctx *c, const double *x, const double *v, int rebuild) {
    if (x) { memcpy(c->x, x, sizeof(double) * 3 * c->n); memcpy(c->xu, x, sizeof(double) * 3 * c->n); wrap_all(c); }
    if (v) memcpy(c->v, v, sizeof(double) * 3 * c->n);
    if (rebuild) rebuild_rows(c);
    compute_f0(c);
}
int64_t orc_get_step(const orc_ctx *c) { return c->step; }
void orc_set_eps(orc_ctx *c, double eps) { c->p.eps_jump = eps; }
/* R-11: 0 = bound held between accepted jumps (default), 1 = re-evaluated at every proposal (Algorithm 4 as printed) */
void orc_set_bound_mode(orc_ctx *c, int every_proposal) { c->bound_every = every_proposal ? 1 : 0; }
void orc_scale_bounds(orc_ctx *c, double f) { c->GM *= f; c->GL *= f; c->G3 *= f; c->GV *= f; c->GV2 *= f; c->GV3 *= f; } /* thinning-invariance pin */
int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
/* run only the C' (and J') half-step at frozen x: used by the rate / drift pins */
void orc_jump_half(orc_ctx *c, double H_ps, int with_accel, int64_t step) {
    jump_phase(c, H_ps, with_accel ? c->f0 : NULL, 1, 2, step, 0);
}
/* single long-range pair gradient F_ij (kcal/mol/A): which 0 Coulomb, 1 LJ */
double orc_fij(const orc_ctx *c, int which, int i, int j, double F[3]) {
    return which == 0 ? fij_coul(c, i, j, F) : fij_lj(c, i, j, F);
}
/* many draws of G~ at one eta (distribution pins): out[k], returns total attempts */
int64_t orc_gtilde_batch(double eta, uint64_t seed, int n, double *out) {
    orc_ctx c;
    memset(&c, 0, sizeof c);
    c.p.seed = seed;
    int64_t tot = 0;
    for (int k = 0; k < n; ++k) {
        uint32_t b = 0;
        int att = 0;
        double mg = 1e300;
        out[k] = orc_gtilde(&c, eta, k, 0, 99, &b, &att, &mg);
        tot += att;
    }
    return tot;
}
/* overwrite velocities only (no list or force refresh) */
void orc_set_vel(orc_ctx *c, const double *v) { memcpy(c->v, v, sizeof(double) * 3 * c->n); }
