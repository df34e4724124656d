/*
 * jump_b200.h -- C ABI of the B200-native JUMP hot path (arXiv 2412.15073).
 *
 * "P:Lnnn" = line nnn of the paper text; "R-n" = reading n in DESIGN.md.
 * Every entry point takes plain pointers and sizes; pointers named d_* are DEVICE
 * pointers, everything else is HOST memory.  No torch types cross this boundary.
 *
 * Sign convention (R-4): every "force" array is a GRADIENT piece, grad U = sum F
 * (P:L59); the physical force is -F.  Units (R-1): Angstrom, fs for dt_fs, 1/ps for
 * gamma, K, g/mol, e, kcal/mol; velocities in Angstrom/ps; gradients in kcal/mol/A.
 *
 * Errors: every int-returning call gives 0 on success or a negative JUMP_E_* code.
 * Device-side flags (row overflow, thinning bound violated, displacement beyond
 * skin/2, non-finite state) are sticky and reported by the next synchronising call
 * (jump_get_*, jump_sync); jump_reset_stats clears them.  Nothing is printed and
 * nothing calls exit().
 */
#ifndef JUMP_B200_H
#define JUMP_B200_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define JUMP_E_ARG (-1)      /* bad argument (n_inner odd, r_short >= r_long, r_long > box/2, ...) */
#define JUMP_E_CUDA (-2)     /* CUDA runtime error, see jump_last_error */
#define JUMP_E_OVERFLOW (-3) /* a neighbour/ring row or the event buffer overflowed its capacity */
#define JUMP_E_BOUND (-4)    /* thinning bound violated: an acceptance probability p > 1 was seen */
#define JUMP_E_SKIN (-5)     /* an atom moved more than its share of the skin within min(3, nlist_every/4) steps of a list
                                build (or with nlist_every = 0): the lists may have missed a pair (R-10c).  Checked on the
                                device at every step; raise skin.  With JUMP_F_LAX_SKIN only jump_stats.max_disp reports it. */
#define JUMP_E_NAN (-6)      /* non-finite position or velocity */

#define JUMP_F_COUL_JUMPS 1u       /* Coulomb tail r_c..r_long by jumps (step C', Alg. 4) */
#define JUMP_F_LJ_JUMPS 2u         /* LJ tail by BPS jumps (step J', Alg. 5); else LJ tail stays in F0 (R-13) */
#define JUMP_F_EVENT_LOG 4u        /* record every proposal (R-18) */
#define JUMP_F_RESPA_PAPER 8u      /* RESPA: bonded inner, short non-bonded + jumps outer */
#define JUMP_F_RESPA_COMPARATOR 16u /* jump_respa_step runs BAOAB-RESPA: outer kick by the long force */

#define JUMP_F_BJAOAJB 64u         /* jump_step runs B J A O A J B instead of C'J' A O A J'C' */
#define JUMP_F_COMBINED 128u       /* with flags 1 | 2: step C' runs ONE mechanism per pair for the whole long pair gradient, Coulomb + LJ
                                      (bound = sum of the two ring bounds), and there is no step J' (R-22) */
#define JUMP_F_LAX_SKIN 32u        /* a displacement beyond skin/2 between list builds is NOT an error (see JUMP_E_SKIN) */

typedef struct jump_ctx jump_ctx; /* opaque, owned by the library */

/* Run parameters, copied at init.  Passages: P:L591-643 (simulation details), R-1..R-15. */
typedef struct {
    int32_t n_atoms;
    int32_t n_inner;     /* RESPA: Delta = n_inner * dt, must be even */
    int32_t eps_mode;    /* 0 = constant epsilon = eps_jump (Alg. 4); 1 = adaptive eps(x) = eps_jump |F_ij(x)| (
                            DESIGN.md R-19), eps_jump finite, in A mol/kcal */
    uint32_t flags;      /* JUMP_F_* */
    int32_t nlist_every; /* P: all lists are rebuilt P steps after their last build at the latest, and -- decided on the
                            device, step by step -- from min(3, P/4) steps after it on as soon as an atom has moved more
                            than its share of the skin since then (R-10c); 0: never after init */
    int32_t pad0;
    uint64_t seed;       /* Philox4x32-10 key (R-15) */
    double box[3];       /* orthorhombic periodic box edges, A */
    double r_short;      /* r_c: chi = 0 at and beyond it */
    double r_switch;     /* h: chi = 1 below r_c - h */
    double r_mid;        /* r_M: outer ring edge (R-10c: rings [r_c-h, r_A), [r_A, r_M), [r_M, r_long));
                            <= 0: r_A (two rings) */
    double r_long;       /* r_E: pairs beyond are neglected */
    double ewald_alpha;  /* alpha of erfc(alpha r)/r; < 0: 3.8 / r_long (R-2) */
    double dt_fs, gamma_per_ps, temperature_K; /* delta, gamma, T */
    double eps_jump;     /* epsilon of the general mechanism (6),(7); +inf: BPS */
    double skin;         /* list skin s (R-10) */
    double cell_edge;    /* minimum edge of the sort grid; <= 0: (r_long + skin) / 4 (R-10) */
    double r_mid_in;     /* r_A: inner ring edge; <= 0: r_short (ring A = the switching zone) */
} jump_params;

/* One proposal of a jump chain (R-18).  ring: 0, 1, 2 = ring A, B, C of a Coulomb chain (step C'), 4, 5, 6 = the same
 * rings of an LJ chain (step J'), -1 = clock expired.  j: the candidate drawn (original index), whether or not it
 * carries a force at the moment. */
typedef struct {
    int32_t step, stream, atom, iter;
    int32_t ring, j, accepted, n_gt;
    float T, p, U, gt;
} jump_event;

typedef struct {
    int64_t proposals, accepts, gt_attempts, rebuilds, expiries;
    double max_p;        /* largest acceptance probability seen (must stay <= 1) */
    double max_g_over_L; /* largest |F_ij| / L seen (must stay <= 1) */
    double max_disp;     /* largest displacement since a list build, A */
    int32_t max_row[6];  /* largest row length seen: short, A, B, (unused), full, LJ-tail */
    int32_t cap_row[6];  /* row capacities */
    int32_t error;       /* sticky device error (0 or JUMP_E_*) */
    int32_t pad;
} jump_stats;

/*
 * Create a context.  All d_* arrays are device memory owned by the caller and borrowed for the
 * context's lifetime; d_pos / d_vel (n_atoms x 3, row-major, original atom order) are updated in
 * place by the step calls, the others are read at init only (copied into the library's own sorted
 * layout).  lj: 4 eps_ij [(s_ij/r)^12 - (s_ij/r)^6] with geometric mixing (R-8).  Bonds k (r-r0)^2,
 * angles k (theta-theta0)^2 with the vertex in the middle of each ijk triple (R-2).  Exclusions as
 * CSR over original indices (R-9); d_excl_ptr may be NULL for none.  cuda_stream: a cudaStream_t
 * (NULL = default stream); all work is enqueued on it.  Builds the sort, all rows and F0(x0).
 */
int jump_init(jump_ctx **out, const jump_params *p, float *d_pos, float *d_vel, const float *d_mass,
              const float *d_charge, const float *d_lj_sigma, const float *d_lj_eps, int32_t n_bonds,
              const int32_t *d_bond_ij, const float *d_bond_k, const float *d_bond_r0, int32_t n_angles,
              const int32_t *d_angle_ijk, const float *d_angle_k, const float *d_angle_t0,
              const int32_t *d_excl_ptr, const int32_t *d_excl_idx, void *cuda_stream);

/* n_steps of the C'J'AOAJ'C' scheme.  Asynchronous. */
int jump_step(jump_ctx *c, int32_t n_steps);
/* n_steps of BAOAB with the unsplit force to r_long.  Asynchronous. */
int baoab_step(jump_ctx *c, int32_t n_steps);
/* n_outer outer steps of JUMP-RESPA, or BAOAB-RESPA with JUMP_F_RESPA_COMPARATOR (R-12). */
int jump_respa_step(jump_ctx *c, int32_t n_outer);

/* NEXT-2 (R-21): the reciprocal part of the Ewald sum as the slow many-body force
 * F_{0,1} = grad(U_rec + U_excl), U_rec = (C/2V) sum_{k != 0, |k| <= k_cut} (4 pi/k^2) exp(-k^2/4 alpha^2) |S(k)|^2,
 * U_excl = -sum_{excluded pairs} C q_i q_j erf(alpha r)/r.  jump_ewald_setup builds the half-space k list on the host
 * (k_cut in 1/A; <= 0: 8 alpha), uploads it and allocates the scratch; *n_k (host, may be NULL) receives the number of
 * vectors.  Needs ewald_alpha != 0; at most 511 vectors per dimension (JUMP_E_ARG otherwise).  Synchronises. */
int jump_ewald_setup(jump_ctx *c, double k_cut, int32_t *n_k);
/* n_outer outer steps of the three-level JUMP-RESPA1: delta = dt_fs (bonded), kappa = n_inner delta
 * (short non-bonded + the jumps), Delta = n_mid kappa (kick by F_{0,1} on both sides); with JUMP_F_RESPA_COMPARATOR
 * BAOAB-RESPA1: the middle level kicks with the short non-bonded gradient, the long pair gradient rides with F_{0,1}
 * (P:L511).  n_mid >= 1.  Asynchronous; JUMP_E_ARG before jump_ewald_setup. */
int jump_respa1_step(jump_ctx *c, int32_t n_outer, int32_t n_mid);
/* U_rec + U_self + U_excl at the current positions, kcal/mol (host double); 0 with no reciprocal vector.  Synchronises. */
int jump_get_slow_energy(jump_ctx *c, double *e_slow);

/* Gradient pieces at the current positions, original atom order, kcal/mol/A, into d_out (n x 3).
 * which: 0 F0 (bonded + short non-bonded), 1 full (unsplit to r_long), 2 long, 3 bonded, 4 short non-bonded,
 * 5 slow (reciprocal Ewald + exclusion correction, after jump_ewald_setup). */
int jump_get_forces(jump_ctx *c, int32_t which, float *d_out);
/* Kinetic energy and the full unsplit potential to r_long, kcal/mol (host doubles). */
int jump_get_energy(jump_ctx *c, double *e_kin, double *e_pot_full);
int jump_get_stats(jump_ctx *c, jump_stats *host_out);
int jump_reset_stats(jump_ctx *c);
/* Copy up to cap logged events (unsorted) to host_buf; *n receives the number logged so far. */
int jump_get_events(jump_ctx *c, jump_event *host_buf, int64_t cap, int64_t *n);
int jump_clear_events(jump_ctx *c);
/* Candidate lists of original atom i as original indices in canonical order (R-10c): which = 0 short list, 1 row A,
 * 2 row B, 3 the cell universe of the atom's home cell (ring C; it holds the atom itself and its excluded partners);
 * 4 full list, 5 LJ-tail list.  Returns the length (or a negative error); at most cap entries are written to host_out. */
int jump_get_row(jump_ctx *c, int32_t which, int32_t atom, int32_t *host_out, int32_t cap);
/* Observables on the device (the paper's evidence is of this kind).
 * jump_get_images: periodic image counters (n x 3 int32, device, original order): the unwrapped position of atom i is
 *   d_pos[i] + image[i] * box, continuous since jump_init (or the last jump_refresh, which resets the counters;
 *   jump_refresh_lazy keeps them); each counter holds +-511 box lengths (beyond that it wraps: a 512-box excursion).  Synchronises the stream.
 * jump_rdf_accumulate: adds to d_hist[n_bins] (device, uint64, caller-owned and zeroed by the caller) the number of
 *   unordered pairs of atoms (lj_only != 0: of LJ carriers, the water oxygens) whose minimum-image distance r at the
 *   current positions is < r_max, in bin floor(r n_bins / r_max); r_max <= box/2, n_bins <= 2048.  Bonded exclusions
 *   are not applied (a geometric histogram).  Asynchronous on the context's stream.  g(r) is
 *   hist / (n_calls * 0.5 N (N-1) / V * shell volume). */
int jump_get_images(jump_ctx *c, int32_t *d_img);
/* Velocity autocorrelation (the velocity spectra of P:L529-531, L583-589 are its cosine transform).  jump_vacf_mark
 * stores the current velocities, by original atom index, as the time origin (asynchronous).  jump_vacf_dot writes
 * *c_out = (1/N_sel) sum_{i in sel} v_i(origin) . v_i(now) in (A/ps)^2 (host double), sel = all atoms or (lj_only != 0) the LJ
 * carriers; fp64 sums in a fixed order.  Synchronises; JUMP_E_ARG before a mark. */
int jump_vacf_mark(jump_ctx *c);
int jump_vacf_dot(jump_ctx *c, int32_t lj_only, double *c_out);
/* Mean-square displacement (the diffusion constants of P:L527, L575-581 are its long-time slope / 6).  jump_msd_mark stores
 * the current UNWRAPPED positions (d_pos + image counters x box, fp64), by original atom index, as the time origin
 * (asynchronous).  jump_msd writes *msd_out = (1/N_sel) sum_{i in sel} |x_i(now) - x_i(origin)|^2 in A^2 (host double), sel
 * as in jump_vacf_dot; fp64 sums in a fixed order.  Synchronises; JUMP_E_ARG before a mark.  A jump_refresh (not
 * jump_refresh_lazy) resets the image counters and with them the continuity of the unwrapped positions. */
int jump_msd_mark(jump_ctx *c);
int jump_msd(jump_ctx *c, int32_t lj_only, double *msd_out);
int jump_rdf_accumulate(jump_ctx *c, int32_t lj_only, double r_max, int32_t n_bins, uint64_t *d_hist);
/* The same sum for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * no context, no cudaMalloc / cudaFree, the per-CTA partial sums in a 256 KiB file-scope device array of the library
 * (held by every GPU that loads the library until the process exits).
 *   d_v_now, d_v_origin  DEVICE, n x 3 packed floats (the layout of d_vel), the same atom order in both
 *   d_select             DEVICE, n int32 (non-zero = atom counts), or NULL = all atoms
 *   d_out                DEVICE, 2 doubles: (1/N_sel) sum_{i in sel} v_i(origin) . v_i(now) (0 if N_sel = 0), and N_sel
 *   stream               cudaStream_t the two kernels are enqueued on (asynchronous; nothing is synchronised)
 * n > JUMP_VACF_STATIC_MAX_ATOMS, n <= 0 or a null array: JUMP_E_ARG, nothing launched; text in
 * jump_vacf_static_last_error() (per host thread).  All calls on a device share the scratch array: calls that overlap
 * on the GPU (different streams without a dependency) race; calls on one stream, or ordered by events, do not.  The
 * array needs no clearing between calls.  jump_vacf_static_setup() takes the array's device address for the CURRENT
 * device (once per device; the first jump_vacf_dot_static on a device does it too -- call it before a graph capture). */
#define JUMP_VACF_STATIC_MAX_ATOMS 4194304
int jump_vacf_static_setup(void);
int jump_vacf_dot_static(int32_t n, const float *d_v_now, const float *d_v_origin, const int32_t *d_select, double *d_out,
                         void *stream);
const char *jump_vacf_static_last_error(void);
/* Bounds as used (R-7, R-10c): G_A, G_B, GV_A, qmax, eps_max, sig_min, sig_max, r_M, G_C, GV_B, GV_C, r_A (G: sup of the
 * long Coulomb gradient per unit charges over a ring, GV: of the long LJ gradient with 4 eps = 1). */
int jump_get_bounds(jump_ctx *c, double out[12]);
/* Lanes that cooperate on one jump chain in the update kernel: 1, 4, 8 or 16; 0 = chosen from the number of atoms so
 * that the grid fills the GPU once (the default).  Every choice runs the same chains with the same random streams
 * (tests compare each against the oracle).  */
int jump_set_lanes(jump_ctx *c, int32_t lanes);
/* Switch JUMP_F_LAX_SKIN on / off after init (an equilibration from a hot start, then a checked production run). */
int jump_set_lax_skin(jump_ctx *c, int32_t on);
/* Re-read d_pos / d_vel after the caller changed them: re-sort, rebuild rows, recompute F0. */
int jump_refresh(jump_ctx *c);
/* The same for a caller that hands the state back after a few steps (host round trips): the rows are kept, and the
 * sorted order with them, when no atom is farther than skin/2 from its position at the last list build -- they are
 * still supersets of the pairs in range (R-10c); otherwise re-sort and rebuild as jump_refresh does.  *rebuilt (may be
 * NULL) receives 0 / 1.  The list-rebuild period of the step calls keeps counting.  F0 is recomputed.  The image
 * counters are KEPT (the trajectory is taken to continue): an atom whose position comes back bit for bit as the library
 * wrote it keeps its fp64 residual as well; for any other the residual restarts at 0 and a coordinate outside [0, L) adds
 * its box lengths to the counter.  Synchronises the stream once (the decision is taken on the host). */
int jump_refresh_lazy(jump_ctx *c, int32_t *rebuilt);
/* Run only the opening jump half-phase C'(H) [then J'(H)] at frozen x with stream ids 1, 2 (pins). */
int jump_half(jump_ctx *c, double H_ps, int32_t with_accel, int64_t step);
/* Wait for the stream; returns the sticky device error if any. */
int jump_sync(jump_ctx *c);
int64_t jump_get_step(const jump_ctx *c);
/* Number of kernels this context launched so far (bench.py's gpu_launches). */
int64_t jump_get_launches(const jump_ctx *c);
/* Measurement (bench.py): with profiling on, every kernel group is bracketed by CUDA events on the context's
 * stream; jump_get_profile waits for the stream and returns the summed milliseconds and the number of bracketed
 * launches (groups) per category: 0 pair-force kernels, 1 bonded, 2 update (jump chains + integrator),
 * 3 sort + row build.  Turning profiling on or off resets the sums. */
int jump_set_profiling(jump_ctx *c, int32_t on);
int jump_get_profile(jump_ctx *c, double ms[4], int64_t count[4]);
/* Ordered entries of row which_row (0 short .. 5) whose current distance is below r_cut: the number of pair
 * terms one pair-force launch over that row evaluates (each unordered pair counts twice). */
int jump_count_pairs(jump_ctx *c, int32_t which_row, double r_cut, int64_t *n_ordered);
const char *jump_last_error(const jump_ctx *c);
void jump_free(jump_ctx *c);

#ifdef __cplusplus
}
#endif
#endif
