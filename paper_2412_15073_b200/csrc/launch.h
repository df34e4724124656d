// launch.h -- host-side launcher prototypes shared by the .cu files of the CUDA path.
#pragma once
#include "common.cuh"

namespace jb {

// A list (re)build is a fixed sequence of kernels.  go == NULL: they run.  go != NULL: they run only if *go == want, i.e.
// if the update kernel of this very step found an atom farther than skin/2 from its build position (R-10c) -- the
// decision is taken on the device, the host enqueues the sequence either way and never waits for it.
struct SortArgs {
    int n;
    SortGrid grid;
    float4 *xs, *vs, *xl;          // state in the current sorted order: read, then overwritten with the new order
    float2 *lj, *mi, *hw;
    int *orig;
    float4 *xs_t, *vs_t, *xl_t;    // scratch of the permutation
    float2 *lj_t, *mi_t, *hw_t;
    int *orig_t;
    float4 *x_build;
    int *sorted_of, *cell_of;
    int *key, *cell_count, *cell_fill, *cell_start, *tmp_orig, *tmp_src;
    int *scan_sums, *scan_offs;   // scratch of the multi-block scan (ncell / 4096 + 2 each)
    Counters *ctr;
    const int *go;
    int want;
};

struct UpdateArgs {
    Phase ph[2];
    const float4 *grad[2];   // gradient of each phase = grad + grad_b (grad_b may be NULL)
    const float4 *grad_b[2];
    int do_aoa;
    float half_dt, c1, c2;  // delta/2 (ps), exp(-gamma delta), sqrt(1 - c1^2)
    unsigned o_step;        // Philox step index of the O part
    const float4 *xs;
    float4 *xs_out;
    float4 *vs;
    float4 *xl_out;  // position residuals x - xs after A-O-A (a second buffer: the chains of other atoms still read xl_all)
    const float2 *mi, *lj;
    const int *orig;
    const float4 *x_build;
    Row rowA, rowB;
    Universe uni;
    SortGrid grid;
    const int *cell_start;
    const float4 *xl_all;   // position residuals (read-only use: ring-edge ties)
    const int *excl_ptr, *excl_idx;   // exclusions by original index (ring C candidates are not filtered at a build)
    Counters *ctr;
    jump_event *events;  // NULL: no log
    long long event_cap;
    int lanes;           // lanes per jump chain (0: chosen from the grid size)
    int trigger;         // 1: a conditional list build follows this launch and this kernel decides whether it runs (R-10c:
                         // list_P steps after the last build, or from list_Q steps after it on when an atom is beyond its share
                         // of the skin); 0: none follows.  A displacement beyond skin/2 that arms nothing is the error ERR_SKIN
    int step_id;         // the stamp it is armed with
    int list_P, list_Q;
};

struct EwaldArgs {   // reciprocal Ewald sum (ewald.cu, R-21)
    int nk, nch;             // half-space k-vectors, atom chunks of the structure-factor pass
    double alpha;
    const int *kpack;        // [nk] packed (nx, ny, nz)
    const double *coefA;     // [nk] A_k = (C/V)(4 pi/k^2) exp(-k^2/4 alpha^2), fp64 from the host
    double2 *part;           // [nch][nk] structure-factor partials
    double2 *W;              // [nk] 2 A_k S(k)
    double *ek;              // [nk] A_k |S(k)|^2
    int nmax[3];             // largest |n| per dimension
    int ntile;               // register-blocked structure-factor pass: 4 x 4 (ny, nz) tiles holding a k-vector (0: not used)
    const int *tiles;        // [ntile] packed (nx, ny0, nz0)
    const int *cube2k;       // [(nmax_x + 1)(2 nmax_y + 1)(2 nmax_z + 1)] cube position -> index in the k list, -1 outside
    float2 *Wt;              // [16][ntile] W in tile order (register-blocked force pass)
    float2 *tabF;            // [n][E] fp32 phase-factor tables (register-blocked force pass)
    double2 *tabD;           // [E][n] fp64 phase-factor tables (NULL: direct sines and cosines), E = sum (nmax + 1)
};

void launch_sort(const SortArgs &a, const Universe &u, unsigned short *uni_cum, cudaStream_t st, int64_t *launches);
int launch_universe_list(const SortGrid &g, const Universe &u, const int *cell_start, int home, int *out, int cap,
                         cudaStream_t st, int64_t *launches);
void launch_build_rows(const Model &m, const SortGrid &g, const Row rows[N_ROWS], float rmax_all, const int *cell_start,
                       const float4 *xs, const float4 *xl, const float2 *lj, const float2 *hw, const int *orig, const int *sorted_of,
                       const int *excl_ptr, const int *excl_idx, Counters *ctr, int *cell_of, float far2, const int *go, int want,
                       cudaStream_t st, int64_t *launches);
int launch_pair(const Model &m, const Row &row, int wC, int wLJ, const float4 *xs, const float2 *lj, float4 *out,
                int accumulate, bool energy, cudaStream_t st, int64_t *launches);
void launch_count_pairs(const Model &m, const Row &row, const float4 *xs, float rc2, unsigned long long *out,
                        cudaStream_t st, int64_t *launches);
void launch_bonded(const Model &m, const Topo &t, const Bonded &b, const float4 *xs, const float4 *xl, const int *sorted_of,
                   float4 *out_bond, cudaStream_t st, int64_t *launches);
void launch_unsort3(int n, const float4 *f, const float4 *f2, const int *orig, float *out, cudaStream_t st, int64_t *launches);
void launch_update(const Model &m, const UpdateArgs &A, bool jumps, cudaStream_t st, int64_t *launches);
void launch_writeback(int n, const float4 *xs, const float4 *vs, const int *orig, float *pos, float *vel, cudaStream_t st,
                      int64_t *launches);
void launch_load(const Model &m, const float *pos, const float *vel, const float *mass, const float *charge,
                 const float *sigma, const float *eps, double kT, double hs_over_wnorm, float4 *xs, float4 *vs, float4 *xl, float2 *lj,
                 float2 *mi, float2 *hw, int *orig, cudaStream_t st, int64_t *launches);
void launch_reload(const Model &m, const float *pos, const float *vel, const int *orig, float4 *xs, float4 *vs,
                   float4 *xl, const float4 *x_build, int *moved, int keep, const float2 *mi, cudaStream_t st, int64_t *launches);
int launch_rdf(const Model &m, const SortGrid &g, int lj_only, double r_max, double r_reach, int n_bins, const int *cell_start,
               const float4 *xs, const float2 *lj, unsigned long long *hist, cudaStream_t st, int64_t *launches);
void launch_msd_mark(const Model &m, const float4 *xs, const float4 *xl, const int *orig, double *x0, cudaStream_t st, int64_t *launches);
void launch_msd_sum(const Model &m, int lj_only, const float4 *xs, const float4 *xl, const int *orig, const float2 *lj, const double *x0,
                    double2 *part, double2 *out, cudaStream_t st, int64_t *launches);
void launch_vacf_mark(int n, const float4 *vs, const int *orig, float4 *v0, cudaStream_t st, int64_t *launches);
void launch_vacf_dot(int n, int lj_only, const float4 *vs, const float4 *v0, const int *orig, const float2 *lj, double2 *part,
                     double2 *out, cudaStream_t st, int64_t *launches);
void launch_images(int n, const float4 *xl, const int *orig, int *out, cudaStream_t st, int64_t *launches);
void launch_kinetic(int n, const float4 *vs, const float2 *mi, double *out, cudaStream_t st, int64_t *launches);
void launch_rec_force(const Model &m, const EwaldArgs &e, const float4 *xs, const float4 *xl, const int *orig,
                      const int *sorted_of, const int *excl_ptr, const int *excl_idx, float4 *out, cudaStream_t st,
                      int64_t *launches);
void launch_rec_energy(const EwaldArgs &e, double *out, cudaStream_t st, int64_t *launches);
int ewald_pack(int nx, int ny, int nz);
int ewald_table_entries_max();

}  // namespace jb
