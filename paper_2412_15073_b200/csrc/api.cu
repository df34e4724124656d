// api.cu -- context, host-side step drivers and the C ABI of include/jump_b200.h.
// The drivers only enqueue kernels on one stream; every arithmetic step of the path runs in the
// kernels of sort_build.cu, forces.cu and update.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <string>
#include <vector>

#include "launch.h"

using namespace jb;

struct jump_ctx {
    jump_params p;
    Model m;
    SortGrid g;
    cudaStream_t st;
    cudaStream_t st2;            // side stream: the bonded kernel runs beside the pair kernel (fork / join by events)
    cudaEvent_t ev_fork, ev_join;
    bool bonded_in_flight;
    int n;
    double kT, dt, alpha, rA, rM, lo;  // ps; lo = max(r_c - h - skin, 0)
    double G[3], GV[3], qmax, eps_max, sig_min, sig_max;   // bounds per ring (R-7, R-10c)
    double qmin_abs;
    double w_max, w_norm;        // mass weights of the skin: w_i = m_i^-1/2 / w_norm, w_norm = mean(m^-1/2) (R-10c)
    Universe uni;                // cell universe of ring C (R-10c)
    unsigned short *uni_cum;
    int *cell_of;
    int lanes;                   // jump_set_lanes
    float c1, c2;
    float *d_pos, *d_vel;  // caller's
    // sorted state (cur) and spare buffers (nxt)
    float4 *xs, *xs_nxt, *vs, *vs_nxt, *xl, *xl_nxt, *x_build;
    float2 *lj, *lj_nxt, *mi, *mi_nxt, *hw, *hw_nxt;   // hw: (skin/2) w_i, split fp64 (R-10c)
    int *orig, *orig_nxt, *sorted_of;
    int *key, *cell_count, *cell_fill, *cell_start, *tmp_orig, *tmp_src, *scan_sums, *scan_offs;
    Row rows[N_ROWS];
    bool row_active[N_ROWS];      // refreshed by every list build
    int64_t row_last_use[N_ROWS];
    bool f0_valid;           // c->f0 / fnb / fbond hold F0 at the current positions
    float4 *fnb, *fbond, *f0, *ftmp, *ftmp2;
    // reciprocal Ewald sum, the slow force of JUMP-RESPA1 (R-21): set up by jump_ewald_setup
    EwaldArgs ew;
    float4 *fslow;
    double *ew_sum;
    double q2sum;            // sum of q_i^2 (self term)
    float4 *vacf_v0;         // velocities at the time origin of the autocorrelation, by original atom index
    double2 *vacf_part;
    double *msd_x0;          // unwrapped positions at the time origin of the mean-square displacement, by original atom index
    double2 *msd_part;
    bool slow_valid;         // fslow holds grad(U_rec + U_excl) at the current positions, in the current sorted order
    int64_t outer1;

    double *ke;
    unsigned long long *pair_count;   // scratch of jump_count_pairs
    int *moved_flag;                  // scratch of jump_refresh_lazy
    int *excl_ptr, *excl_idx;
    Topo topo;
    Bonded bonded;               // small molecules (one thread each) + atoms of larger components (forces.cu)
    std::vector<void *> owned;  // everything to cudaFree
    Counters *ctr;
    jump_event *events;
    long long event_cap;
    int64_t step, outer, launches;
    int sticky;
    std::string err;
    // optional per-category kernel timing with CUDA events on the launch stream (bench.py's roofline leg)
    bool prof;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_pend[4], prof_free;
    double prof_ms[4];
    int64_t prof_n[4];
};
enum { PROF_PAIR = 0, PROF_BONDED = 1, PROF_UPDATE = 2, PROF_BUILD = 3 };
// a gradient held as the sum of two arrays (b may be NULL): the fused F0 launch leaves pair and bonded parts apart
struct GradRef { const float4 *a, *b; };
static GradRef gr(const float4 *a, const float4 *b = nullptr) { return GradRef{a, b}; }

static void prof_begin(jump_ctx *c, int cat) {
    if (!c->prof) return;
    std::pair<cudaEvent_t, cudaEvent_t> ev;
    if (!c->prof_free.empty()) { ev = c->prof_free.back(); c->prof_free.pop_back(); }
    else { cudaEventCreate(&ev.first); cudaEventCreate(&ev.second); }
    cudaEventRecord(ev.first, c->st);
    c->prof_pend[cat].push_back(ev);
}
static void prof_end(jump_ctx *c, int cat) {
    if (!c->prof) return;
    cudaEventRecord(c->prof_pend[cat].back().second, c->st);
}
static void prof_collect(jump_ctx *c) {
    cudaStreamSynchronize(c->st);
    for (int k = 0; k < 4; ++k) {
        for (auto &ev : c->prof_pend[k]) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, ev.first, ev.second) == cudaSuccess) { c->prof_ms[k] += ms; c->prof_n[k]++; }
            c->prof_free.push_back(ev);
        }
        c->prof_pend[k].clear();
    }
}

#define CK(call)                                                                          \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess) {                                                          \
            c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                  \
            return JUMP_E_CUDA;                                                           \
        }                                                                                 \
    } while (0)

template <class T>
static int dalloc(jump_ctx *c, T **p, size_t count) {
    void *q = nullptr;
    CK(cudaMalloc(&q, std::max<size_t>(count, 1) * sizeof(T)));
    c->owned.push_back(q);
    *p = (T *)q;
    return 0;
}
template <class T>
static int dupload(jump_ctx *c, T **p, const std::vector<T> &h) {
    int r = dalloc(c, p, h.size());
    if (r) return r;
    if (!h.empty()) CK(cudaMemcpyAsync(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));
    return 0;
}
template <class T>
static int ddownload(jump_ctx *c, std::vector<T> &h, const T *d, size_t count) {
    h.resize(count);
    if (count) CK(cudaMemcpyAsync(h.data(), d, count * sizeof(T), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return 0;
}

// ---- bounds L (R-7): sup of the long-part radial derivative on a dense grid, times (1 + 1e-6) ---------------
static void chi_host(double r, double rc, double h, double *chi, double *dchi) {
    double u = (r - (rc - h)) / h;
    if (u <= 0.0) { *chi = 1.0; *dchi = 0.0; return; }
    if (u >= 1.0) { *chi = 0.0; *dchi = 0.0; return; }
    *chi = 1.0 - u * u * u * (10.0 - 15.0 * u + 6.0 * u * u);
    *dchi = -30.0 * u * u * (1.0 - u) * (1.0 - u) / h;
}
static double sup_long(const jump_ctx *c, double lo, double hi, double step, bool coul, double sig) {
    if (!(hi > lo)) return 0.0;
    const double rc = c->p.r_short, h = c->p.r_switch, al = c->alpha;
    double best = 0.0;
    long K = (long)std::floor((hi - lo) / step);
    for (long k = 0; k <= K + 1; ++k) {
        double r = (k <= K) ? lo + step * (double)k : hi;
        if (r > hi) r = hi;
        double u, du;
        if (coul) {  // unit charges: u = C erfc(alpha r)/r
            double e = std::erfc(al * r);
            u = kCoulomb * e / r;
            du = -kCoulomb * (e / (r * r) + 2.0 * al / std::sqrt(M_PI) * std::exp(-al * al * r * r) / r);
        } else {  // 4 eps = 1
            double s = sig / r, s6 = s * s * s * s * s * s, s12 = s6 * s6;
            u = s12 - s6;
            du = (-12.0 * s12 + 6.0 * s6) / r;
        }
        double chi, dchi;
        chi_host(r, rc, h, &chi, &dchi);
        best = std::max(best, std::fabs((1.0 - chi) * du - dchi * u));
    }
    return best * (1.0 + 1e-6);
}
static void compute_bounds(jump_ctx *c, const std::vector<float> &q, const std::vector<float> &sig,
                           const std::vector<float> &eps) {
    c->qmax = 0.0; c->eps_max = 0.0; c->sig_min = 1e300; c->sig_max = 0.0; c->qmin_abs = 1e300;
    for (int i = 0; i < c->n; ++i) {
        c->qmax = std::max(c->qmax, std::fabs((double)q[i]));
        c->qmin_abs = std::min(c->qmin_abs, std::fabs((double)q[i]));
        if (eps[i] > 0.f) {
            c->eps_max = std::max(c->eps_max, (double)eps[i]);
            c->sig_min = std::min(c->sig_min, (double)sig[i]);
            c->sig_max = std::max(c->sig_max, (double)sig[i]);
        }
    }
    if (c->eps_max == 0.0) c->sig_min = c->sig_max = 0.0;
    // R-10c: ring Y holds the pairs whose current distance lies in it, so its bound is the sup over the ring itself
    const double rlo = c->p.r_short - c->p.r_switch, rE = c->p.r_long;
    const double eA = std::min(std::max(c->rA, rlo), rE), eM = std::min(std::max(c->rM, eA), rE);
    const double edge[4] = {rlo, eA, eM, rE};
    const int NS = (c->sig_max > c->sig_min) ? 65 : 1;
    for (int y = 0; y < 3; ++y) {
        c->G[y] = sup_long(c, edge[y], edge[y + 1], 1e-4, true, 0.0);
        c->GV[y] = 0.0;
        if (c->sig_max > 0.0)
            for (int k = 0; k < NS; ++k) {
                double sg = NS == 1 ? c->sig_min : c->sig_min + (c->sig_max - c->sig_min) * (double)k / (double)(NS - 1);
                c->GV[y] = std::max(c->GV[y], sup_long(c, edge[y], edge[y + 1], 1e-4, false, sg));
            }
    }
}

static int round32(double x) { return (int)(((long long)std::ceil(x) + 31) / 32 * 32); }

static int alloc_row(jump_ctx *c, int k) {
    Row &R = c->rows[k];
    if (R.idx) return 0;
    int r = dalloc(c, &R.idx, (size_t)c->n * R.cap);
    if (r) return r;
    r = dalloc(c, &R.cnt, (size_t)c->n);
    if (r) return r;
    CK(cudaMemsetAsync(R.cnt, 0, sizeof(int) * c->n, c->st));
    R.enabled = 1;
    return 0;
}

// Build the given rows in one launch from the positions of the last sort (x_build: what the cell table describes and
// the displacement check refers to; at the sort itself they are the current positions).  go / want: see SortArgs.
static int build_rows(jump_ctx *c, const bool want[N_ROWS], const int *go, int stamp) {
    Row sel[N_ROWS];
    bool any = false;
    double rmax = 0.0;
    for (int k = 0; k < N_ROWS; ++k) {
        sel[k] = c->rows[k];
        if (!(want[k] && c->rows[k].enabled)) sel[k].enabled = 0;
        if (sel[k].enabled) { any = true; rmax = std::max(rmax, (double)std::sqrt(sel[k].r2max)); }
    }
    if (!any) return 0;
    prof_begin(c, PROF_BUILD);
    launch_build_rows(c->m, c->g, sel, (float)rmax, c->cell_start, c->x_build, c->xl, c->lj, c->hw, c->orig,
                      c->sorted_of, c->excl_ptr, c->excl_idx, c->ctr, (sel[ROW_A].enabled ? c->cell_of : nullptr),
                      (float)std::pow(std::max(c->rM - 2.0 * c->p.skin * c->w_max, 0.0), 2), go, stamp, c->st, &c->launches);
    prof_end(c, PROF_BUILD);
    CK(cudaGetLastError());
    return 0;
}

// Sort + universe sums + every active row.  conditional: the kernels run only if the update kernel of this step armed
// them (an atom farther than skin/2 from its build position, R-10c); the host never learns which way it went, so the
// sorted state is permuted through scratch arrays and copied back (no pointer swap) and sorts are counted on the device.
static int resort_and_build(jump_ctx *c, bool conditional) {
    const int *go = conditional ? &c->ctr->go_step : nullptr;
    const int stamp = (int)c->step;
    SortArgs a;
    a.n = c->n; a.grid = c->g;
    a.xs = c->xs; a.vs = c->vs; a.xl = c->xl; a.lj = c->lj; a.mi = c->mi; a.hw = c->hw; a.orig = c->orig;
    a.xs_t = c->xs_nxt; a.vs_t = c->vs_nxt; a.xl_t = c->xl_nxt; a.lj_t = c->lj_nxt; a.mi_t = c->mi_nxt; a.hw_t = c->hw_nxt; a.orig_t = c->orig_nxt;
    a.sorted_of = c->sorted_of; a.x_build = c->x_build; a.cell_of = c->cell_of;
    a.key = c->key; a.cell_count = c->cell_count; a.cell_fill = c->cell_fill; a.cell_start = c->cell_start;
    a.tmp_orig = c->tmp_orig; a.tmp_src = c->tmp_src; a.scan_sums = c->scan_sums; a.scan_offs = c->scan_offs; a.ctr = c->ctr;
    a.go = go; a.want = stamp;
    prof_begin(c, PROF_BUILD);
    launch_sort(a, c->uni, c->uni_cum, c->st, &c->launches);   // (with the running sums of the universe of every cell, ring C, R-10c)
    prof_end(c, PROF_BUILD);
    CK(cudaGetLastError());
    c->slow_valid = false;   // (the sorted order may have changed)
    // rows that nobody has read for a while leave the active set (they are built again on demand)
    for (int k = 0; k < N_ROWS; ++k)
        if (c->row_active[k] && c->step - c->row_last_use[k] > 36) c->row_active[k] = false;
    return build_rows(c, c->row_active, go, stamp);
}

// every read of a row goes through here: allocate on first use; a row outside the active set is built now (from the
// positions of the last sort) and joins it: from then on every list build refreshes it
static int need_rows(jump_ctx *c, std::initializer_list<int> ks) {
    bool want[N_ROWS] = {false, false, false, false, false, false};
    bool stale = false;
    for (int k : ks) {
        int r = alloc_row(c, k);
        if (r) return r;
        c->row_last_use[k] = c->step;
        want[k] = !c->row_active[k];
        stale |= want[k];
        c->row_active[k] = true;
    }
    return stale ? build_rows(c, want, nullptr, 0) : 0;
}
static int need_row(jump_ctx *c, int k) { return need_rows(c, {k}); }

static int pair(jump_ctx *c, int row, int wC, int wLJ, float4 *out, int accumulate, bool energy) {
    int r = need_row(c, row);
    if (r) return r;
    prof_begin(c, PROF_PAIR);
    r = launch_pair(c->m, c->rows[row], wC, wLJ, c->xs, c->lj, out, accumulate, energy, c->st, &c->launches);
    prof_end(c, PROF_PAIR);
    if (r) { c->err = "no pair kernel for this (Coulomb, LJ) weight combination"; return JUMP_E_ARG; }
    return 0;
}
static bool lj_jumps(const jump_ctx *c) { return (c->p.flags & JUMP_F_LJ_JUMPS) != 0; }
static bool coul_jumps(const jump_ctx *c) { return (c->p.flags & JUMP_F_COUL_JUMPS) != 0; }

// bonded gradient at the current positions into c->fbond (the one evaluation every path uses: steps and observers)
static int bonded_eval(jump_ctx *c, cudaStream_t st) {
    launch_bonded(c->m, c->topo, c->bonded, c->xs, c->xl, c->sorted_of, c->fbond, st, &c->launches);
    CK(cudaGetLastError());
    return 0;
}
// F0 = bonded + short non-bonded (R-13: the LJ tail stays in F0 when LJ jumps are off)
static int compute_short_nb(jump_ctx *c, float4 *out, bool energy = false) {
    int r;
    if (lj_jumps(c)) r = pair(c, ROW_S, W_SHORT, W_SHORT, out, 0, energy);
    else {
        r = pair(c, ROW_S, W_SHORT, W_FULL, out, 0, energy);
        if (!r) r = pair(c, ROW_W, W_NONE, W_FULL, out, 1, energy);
    }
    if (r) return r;
    CK(cudaGetLastError());
    return 0;
}
static int bonded_only(jump_ctx *c) {  // fbond at the current positions
    prof_begin(c, PROF_BONDED);
    int r = bonded_eval(c, c->st);
    prof_end(c, PROF_BONDED);
    return r;
}
// the same on the side stream: fork after everything enqueued so far, join_bonded() before fbond is read.
// The bonded kernels then overlap the pair kernel instead of preceding it.
static int bonded_fork(jump_ctx *c) {
    CK(cudaEventRecord(c->ev_fork, c->st));
    CK(cudaStreamWaitEvent(c->st2, c->ev_fork, 0));
    if (c->prof) {   // bracket on the side stream (the categories then overlap in time)
        std::pair<cudaEvent_t, cudaEvent_t> ev;
        if (!c->prof_free.empty()) { ev = c->prof_free.back(); c->prof_free.pop_back(); }
        else { cudaEventCreate(&ev.first); cudaEventCreate(&ev.second); }
        cudaEventRecord(ev.first, c->st2);
        c->prof_pend[PROF_BONDED].push_back(ev);
    }
    int r = bonded_eval(c, c->st2);
    if (c->prof) cudaEventRecord(c->prof_pend[PROF_BONDED].back().second, c->st2);
    if (r) return r;
    CK(cudaEventRecord(c->ev_join, c->st2));
    c->bonded_in_flight = true;
    return 0;
}
static int bonded_join(jump_ctx *c) {
    if (!c->bonded_in_flight) return 0;
    CK(cudaStreamWaitEvent(c->st, c->ev_join, 0));
    c->bonded_in_flight = false;
    return 0;
}
// F0 kept as fnb + fbond (the integrator adds the two)
static int compute_f0(jump_ctx *c) {
    int r = bonded_fork(c);
    if (r) return r;
    r = compute_short_nb(c, c->fnb);
    if (r) return r;
    c->f0_valid = true;
    return bonded_join(c);
}
static GradRef gr_f0(const jump_ctx *c) { return gr(c->fnb, c->fbond); }
static int ensure_f0(jump_ctx *c) { return c->f0_valid ? 0 : compute_f0(c); }
// unsplit force to r_long as ftmp2 + fbond (BAOAB comparator); invalidates F0
static int compute_full_split(jump_ctx *c) {
    int r = bonded_fork(c);
    if (r) return r;
    if ((r = pair(c, ROW_F, W_FULL, W_FULL, c->ftmp2, 0, false))) return r;
    CK(cudaGetLastError());
    c->f0_valid = false;
    return bonded_join(c);
}
static GradRef gr_full(const jump_ctx *c) { return gr(c->ftmp2, c->fbond); }
// long part of the pair gradient (comparators only): the (1 - chi) weights over the full list
static int compute_long(jump_ctx *c, float4 *out) {
    int wLJ = lj_jumps(c) ? W_LONG : W_NONE;
    int r = pair(c, ROW_F, W_LONG, wLJ, out, 0, false);
    if (r) return r;
    CK(cudaGetLastError());
    return 0;
}
static int compute_full(jump_ctx *c, bool energy) {  // unsplit to r_long (ftmp2) + bonded (fbond), observers
    int r = pair(c, ROW_F, W_FULL, W_FULL, c->ftmp2, 0, energy);
    if (r) return r;
    CK(cudaGetLastError());
    c->f0_valid = false;
    return bonded_only(c);
}

// ---- step drivers --------------------------------------------------------------------------------------
static Phase ph_none() { Phase p; memset(&p, 0, sizeof p); return p; }
static Phase ph_kick(double H) { Phase p = ph_none(); p.kind = 1; p.H = (float)H; p.use_grad = 1; return p; }
static Phase ph_jump(const jump_ctx *c, double H, bool grad, bool reverse, int sC, int sJ, int64_t step) {
    Phase p = ph_none();
    p.kind = 2; p.H = (float)H; p.use_grad = grad ? 1 : 0; p.reverse = reverse ? 1 : 0;
    p.coul = coul_jumps(c) ? 1 : 0; p.lj = (lj_jumps(c) && !c->m.combined) ? 1 : 0;   // R-22: no J' under the combined mechanism
    p.streamC = sC; p.streamJ = sJ; p.step = (unsigned)step;
    return p;
}

// up to two velocity half-phases, then (aoa) A O A + wrap, step counter and the scheduled rebuild (C.3 steps 3-6)
static int run_update(jump_ctx *c, const Phase &p0, GradRef g0, const Phase &p1, GradRef g1, bool aoa) {
    UpdateArgs A;
    memset(&A, 0, sizeof A);
    A.ph[0] = p0; A.ph[1] = p1; A.grad[0] = g0.a; A.grad[1] = g1.a; A.grad_b[0] = g0.b; A.grad_b[1] = g1.b;
    if (!g0.a) A.ph[0].use_grad = 0;
    if (!g1.a) A.ph[1].use_grad = 0;
    A.do_aoa = aoa ? 1 : 0;
    A.half_dt = (float)(0.5 * c->dt); A.c1 = c->c1; A.c2 = c->c2; A.o_step = (unsigned)c->step;
    A.xs = c->xs; A.xs_out = c->xs_nxt; A.vs = c->vs; A.xl_out = c->xl_nxt; A.mi = c->mi; A.lj = c->lj; A.orig = c->orig; A.x_build = c->x_build;
    A.rowA = c->rows[ROW_A]; A.rowB = c->rows[ROW_B];
    A.uni = c->uni; A.grid = c->g; A.cell_start = c->cell_start; A.xl_all = c->xl; A.excl_ptr = c->excl_ptr; A.excl_idx = c->excl_idx;
    A.lanes = c->lanes;
    // R-10c list schedule, counted from the last build: P = nlist_every steps after it at the latest; from Q = min(3, P/4)
    // steps after it on as soon as an atom has used up its share of the skin (before that: the error JUMP_E_SKIN).  The update kernel
    // decides (only the device knows when the last build was); the list kernels are enqueued behind it at every step.
    const int P = c->p.nlist_every;
    const int64_t next = c->step + 1;
    const bool will_check = aoa && P > 0;
    A.trigger = will_check ? 1 : 0;
    A.step_id = (int)next;
    A.list_P = P; A.list_Q = P >= 12 ? 3 : (P >= 4 ? P / 4 : 1);
    A.ctr = c->ctr; A.events = (c->p.flags & JUMP_F_EVENT_LOG) ? c->events : nullptr; A.event_cap = c->event_cap;
    bool jumps = (p0.kind == 2 || p1.kind == 2) && (coul_jumps(c) || lj_jumps(c));
    if (jumps) {
        int r = need_rows(c, {ROW_A, ROW_B});
        if (r) return r;
        A.rowA = c->rows[ROW_A]; A.rowB = c->rows[ROW_B];
    }
    prof_begin(c, PROF_UPDATE);
    launch_update(c->m, A, jumps, c->st, &c->launches);
    prof_end(c, PROF_UPDATE);
    CK(cudaGetLastError());
    if (aoa) {
        std::swap(c->xs, c->xs_nxt);
        std::swap(c->xl, c->xl_nxt);
        c->f0_valid = false;
        c->slow_valid = false;
        c->step++;
        if (will_check) return resort_and_build(c, true);
    }
    return 0;
}
static int writeback(jump_ctx *c) {
    launch_writeback(c->n, c->xs, c->vs, c->orig, c->d_pos, c->d_vel, c->st, &c->launches);
    CK(cudaGetLastError());
    return 0;
}
static int poll_error(jump_ctx *c) {  // sticky device flags -> error code
    Counters h;
    CK(cudaMemcpyAsync(&h, c->ctr, sizeof h, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    if (h.err & ERR_NAN) c->sticky = JUMP_E_NAN;
    else if (h.err & (ERR_OVERFLOW | ERR_EVENTS)) c->sticky = JUMP_E_OVERFLOW;
    else if (h.err & ERR_BOUND) c->sticky = JUMP_E_BOUND;
    else if ((h.err & ERR_SKIN) && !(c->p.flags & JUMP_F_LAX_SKIN)) c->sticky = JUMP_E_SKIN;
    if (c->sticky && c->err.empty()) c->err = "device error flags " + std::to_string(h.err);
    return c->sticky;
}

extern "C" int jump_step(jump_ctx *c, int32_t n_steps) {
    if (!c || n_steps < 0) return JUMP_E_ARG;
    if (n_steps == 0) return 0;
    const double H = 0.5 * c->dt;
    const bool bj = (c->p.flags & JUMP_F_BJAOAJB) != 0;
    int r0 = ensure_f0(c);
    if (r0) return r0;
    for (int s = 0; s < n_steps; ++s) {
        int64_t st = c->step;
        Phase open = ph_jump(c, H, true, false, 1, 2, st);
        Phase close_prev = s > 0 ? ph_jump(c, H, true, true, 4, 3, st - 1) : ph_none();
        if (bj) { open.bkick = 1; close_prev.bkick = 2; }   // B J A O A J B
        int r = run_update(c, close_prev, gr_f0(c), open, gr_f0(c), true);
        if (r) return r;
        r = compute_f0(c);
        if (r) return r;
    }
    Phase close_last = ph_jump(c, H, true, true, 4, 3, c->step - 1);
    if (bj) close_last.bkick = 2;
    int r = run_update(c, close_last, gr_f0(c), ph_none(), gr(nullptr), false);
    if (r) return r;
    return writeback(c);
}

extern "C" int baoab_step(jump_ctx *c, int32_t n_steps) {
    if (!c || n_steps < 0) return JUMP_E_ARG;
    if (n_steps == 0) return 0;
    const double H = 0.5 * c->dt;
    int r = compute_full_split(c);
    if (r) return r;
    for (int s = 0; s < n_steps; ++s) {
        r = run_update(c, s > 0 ? ph_kick(H) : ph_none(), gr_full(c), ph_kick(H), gr_full(c), true);
        if (r) return r;
        r = compute_full_split(c);
        if (r) return r;
    }
    r = run_update(c, ph_kick(H), gr_full(c), ph_none(), gr(nullptr), false);
    if (r) return r;
    return writeback(c);  // F0 is recomputed on demand (f0_valid)
}

// n_outer outer steps of the two-level scheme (R-12).  long_in_outer: the comparator's kick carries the long pair
// gradient (two-level BAOAB-RESPA); false when a third level carries it (BAOAB-RESPA1).  paper: bonded inner,
// short non-bonded (+ jumps) outer.
static int respa_outer_steps(jump_ctx *c, int n_outer, bool paper, bool long_in_outer) {
    const int n = c->p.n_inner;
    const double D = n * c->dt, H = 0.5 * c->dt;
    const bool cmp = (c->p.flags & JUMP_F_RESPA_COMPARATOR) != 0;
    int r = ensure_f0(c);
    if (r) return r;
    for (int o = 0; o < n_outer; ++o) {
        Phase outer[2];
        GradRef gout[2];
        for (int half = 0; half < 2; ++half) {
            if (half == 1) {  // inner loop: n x BAOAB_delta with F_in; the first opening kick rides with outer[0]
                for (int s = 0; s < n; ++s) {
                    GradRef fin = paper ? gr(c->fbond) : gr_f0(c);
                    if (s == 0) r = run_update(c, outer[0], gout[0], ph_kick(H), fin, true);
                    else r = run_update(c, ph_kick(H), fin, ph_kick(H), fin, true);
                    if (r) return r;
                    r = paper ? bonded_only(c) : compute_f0(c);
                    if (r) return r;
                }
                if (paper) { r = compute_f0(c); if (r) return r; }
            }
            if (cmp) {  // BAOAB-RESPA: v <- v - (Delta/2) M^-1 F_long
                float4 *fl = half == 0 ? c->ftmp : c->ftmp2;
                int acc = 0;
                if (long_in_outer) {
                    r = compute_long(c, fl);
                    if (r) return r;
                    acc = 1;
                }
                if (paper) {  // + short non-bonded
                    r = pair(c, ROW_S, W_SHORT, lj_jumps(c) ? W_SHORT : W_FULL, fl, acc, false);
                    if (!r && !lj_jumps(c)) r = pair(c, ROW_W, W_NONE, W_FULL, fl, 1, false);
                    if (r) return r;
                    CK(cudaGetLastError());
                    acc = 1;
                }
                outer[half] = acc ? ph_kick(0.5 * D) : ph_none();
                gout[half] = gr(fl);
            } else {
                gout[half] = gr(paper ? c->fnb : nullptr);
                outer[half] = half == 0 ? ph_jump(c, 0.5 * D, paper, false, 5, 6, c->outer)
                                        : ph_jump(c, 0.5 * D, paper, true, 8, 7, c->outer);
            }
        }
        GradRef fin = paper ? gr(c->fbond) : gr_f0(c);
        r = run_update(c, ph_kick(H), fin, outer[1], gout[1], false);
        if (r) return r;
        c->outer++;
    }
    return 0;
}
extern "C" int jump_respa_step(jump_ctx *c, int32_t n_outer) {
    if (!c || n_outer < 0) return JUMP_E_ARG;
    int r = respa_outer_steps(c, n_outer, (c->p.flags & JUMP_F_RESPA_PAPER) != 0, true);
    if (r) return r;
    return writeback(c);
}

// ---- NEXT-2: reciprocal Ewald sum as the slow force, three-level JUMP-RESPA1 (R-21) ---------------------------
extern "C" int jump_ewald_setup(jump_ctx *c, double k_cut, int32_t *n_k) {
    if (!c) return JUMP_E_ARG;
    if (!(c->alpha > 0.0)) { c->err = "the reciprocal sum needs ewald_alpha > 0"; return JUMP_E_ARG; }
    if (!(k_cut > 0.0)) k_cut = 8.0 * c->alpha;   // exp(-k^2/4 alpha^2) = e^-16 = 1.1e-7, the size of erfc(3.8) (R-2)
    const double two_pi = 6.283185307179586476925;
    const double V = c->p.box[0] * c->p.box[1] * c->p.box[2];
    int nmax[3];
    for (int d = 0; d < 3; ++d) {
        nmax[d] = (int)std::floor(k_cut * c->p.box[d] / two_pi);
        if (nmax[d] > 511) { c->err = "k_cut needs more than 511 reciprocal vectors per dimension"; return JUMP_E_ARG; }
    }
    std::vector<int> kp;
    std::vector<double> cA;
    for (int nx = 0; nx <= nmax[0]; ++nx)
        for (int ny = (nx == 0 ? 0 : -nmax[1]); ny <= nmax[1]; ++ny)
            for (int nz = ((nx == 0 && ny == 0) ? 1 : -nmax[2]); nz <= nmax[2]; ++nz) {
                const double kx = two_pi * nx / c->p.box[0], ky = two_pi * ny / c->p.box[1], kz = two_pi * nz / c->p.box[2];
                const double k2 = kx * kx + ky * ky + kz * kz;
                if (k2 > k_cut * k_cut) continue;
                kp.push_back(ewald_pack(nx, ny, nz));
                cA.push_back((kCoulomb / V) * (4.0 * 3.14159265358979323846 / k2) * std::exp(-k2 / (4.0 * c->alpha * c->alpha)));
            }
    EwaldArgs e;
    memset(&e, 0, sizeof e);
    e.nk = (int)kp.size();
    e.nch = std::max(1, std::min(16, c->n / 512));   // atom chunks of the structure-factor pass (more CTAs, fixed order)
    e.alpha = c->alpha;
    int r;
    int *dk = nullptr;
    double *dA = nullptr;
    if ((r = dupload(c, &dk, kp)) || (r = dupload(c, &dA, cA))) return r;
    e.kpack = dk; e.coefA = dA;
    if ((r = dalloc(c, &e.W, (size_t)e.nk)) || (r = dalloc(c, &e.ek, (size_t)e.nk))) return r;
    // factorised phase tables for the structure-factor pass when a tile of them fits the shared memory;
    // JUMP_B200_EWALD_DIRECT=1 forces the direct form
    int used[3] = {0, 0, 0};
    for (size_t t = 0; t < kp.size(); ++t) {
        const int w = kp[t];
        const int nn[3] = {(w & 1023) - 512, ((w >> 10) & 1023) - 512, ((w >> 20) & 1023) - 512};
        for (int d = 0; d < 3; ++d) used[d] = std::max(used[d], std::abs(nn[d]));
    }
    for (int d = 0; d < 3; ++d) e.nmax[d] = used[d];
    const int E = used[0] + used[1] + used[2] + 3;
    const char *direct = getenv("JUMP_B200_EWALD_DIRECT");
    if (e.nk > 0 && E <= ewald_table_entries_max() && !(direct && atoi(direct) != 0)) {
        if ((r = dalloc(c, &e.tabD, (size_t)E * c->n))) return r;
        // tiles of the register-blocked pass (JUMP_B200_EWALD_BLOCKED=0: one term per thread instead)
        const char *blk = getenv("JUMP_B200_EWALD_BLOCKED");
        if (!(blk && atoi(blk) == 0)) {
            const int Y = 2 * used[1] + 1, Z = 2 * used[2] + 1;
            std::vector<int> cube((size_t)(used[0] + 1) * Y * Z, -1), tiles;
            for (size_t t = 0; t < kp.size(); ++t) {
                const int w = kp[t];
                const int nx = (w & 1023) - 512, ny = ((w >> 10) & 1023) - 512, nz = ((w >> 20) & 1023) - 512;
                cube[((size_t)nx * Y + (ny + used[1])) * Z + (nz + used[2])] = (int)t;
            }
            for (int nx = 0; nx <= used[0]; ++nx)
                for (int ny0 = -used[1]; ny0 <= used[1]; ny0 += 4)
                    for (int nz0 = -used[2]; nz0 <= used[2]; nz0 += 4) {
                        bool any = false;
                        for (int u = 0; u < 4 && !any; ++u)
                            for (int v = 0; v < 4 && !any; ++v) {
                                const int ny = ny0 + u, nz = nz0 + v;
                                if (ny <= used[1] && nz <= used[2]) any = cube[((size_t)nx * Y + (ny + used[1])) * Z + (nz + used[2])] >= 0;
                            }
                        if (any) tiles.push_back(ewald_pack(nx, ny0, nz0));
                    }
            int *dt = nullptr, *dc = nullptr;
            if ((r = dupload(c, &dt, tiles)) || (r = dupload(c, &dc, cube))) return r;
            e.tiles = dt; e.cube2k = dc; e.ntile = (int)tiles.size();
            if ((r = dalloc(c, &e.Wt, (size_t)16 * e.ntile)) || (r = dalloc(c, &e.tabF, (size_t)E * c->n))) return r;
            // fewer threads than k-vectors: atom chunks fill the GPU -- one wave of CTAs (4 per SM at 128 registers)
            int dev = 0, sms = 148;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            const int nblk = (e.ntile + 127) / 128;
            e.nch = std::max(1, std::min(std::max(1, c->n / 64), (4 * sms) / std::max(nblk, 1)));
        }
    }
    if ((r = dalloc(c, &e.part, (size_t)e.nch * e.nk))) return r;   // (after the pass and its number of atom chunks are chosen)
    if (!c->fslow && (r = dalloc(c, &c->fslow, (size_t)c->n))) return r;
    if (!c->ew_sum && (r = dalloc(c, &c->ew_sum, 1))) return r;
    std::vector<float4> hx;
    if ((r = ddownload(c, hx, (const float4 *)c->xs, c->n))) return r;
    c->q2sum = 0.0;
    for (const float4 &v : hx) c->q2sum += (double)v.w * (double)v.w;
    c->ew = e;
    c->slow_valid = false;
    if (n_k) *n_k = e.nk;
    return 0;
}
static int compute_slow(jump_ctx *c) {
    if (c->slow_valid) return 0;
    if (c->ew.nk <= 0) {
        if (!c->fslow) { c->err = "jump_ewald_setup has not been called"; return JUMP_E_ARG; }
        CK(cudaMemsetAsync(c->fslow, 0, sizeof(float4) * c->n, c->st));   // no reciprocal vector: the slow force is off
    } else {
        launch_rec_force(c->m, c->ew, c->xs, c->xl, c->orig, c->sorted_of, c->excl_ptr, c->excl_idx, c->fslow, c->st, &c->launches);
    }
    CK(cudaGetLastError());
    c->slow_valid = true;
    return 0;
}
// Three levels delta, kappa = n_inner delta, Delta = n_mid kappa: the two-level scheme in its paper
// placement between kicks by the slow gradient; comparator: the long pair gradient rides with it.
extern "C" int jump_respa1_step(jump_ctx *c, int32_t n_outer, int32_t n_mid) {
    if (!c || n_outer < 0 || n_mid < 1) return JUMP_E_ARG;
    if (!c->fslow) { c->err = "jump_ewald_setup has not been called"; return JUMP_E_ARG; }
    const bool cmp = (c->p.flags & JUMP_F_RESPA_COMPARATOR) != 0;
    const double D = (double)n_mid * c->p.n_inner * c->dt;
    int r = ensure_f0(c);
    if (r) return r;
    for (int o = 0; o < n_outer; ++o) {
        for (int half = 0; half < 2; ++half) {
            if (half == 1 && (r = respa_outer_steps(c, n_mid, true, false))) return r;
            if ((r = compute_slow(c))) return r;
            const float4 *fl = nullptr;
            if (cmp) {
                if ((r = compute_long(c, c->ftmp))) return r;
                fl = c->ftmp;
            }
            if ((r = run_update(c, ph_kick(0.5 * D), gr(c->fslow, fl), ph_none(), gr(nullptr), false))) return r;
        }
        c->outer1++;
    }
    return writeback(c);
}
// U_rec + U_self + U_excl at the current positions, kcal/mol (0 when no reciprocal vector is set up)
extern "C" int jump_get_slow_energy(jump_ctx *c, double *e_slow) {
    if (!c || !e_slow) return JUMP_E_ARG;
    *e_slow = 0.0;
    if (c->ew.nk <= 0) return 0;
    int r;
    c->slow_valid = false;
    if ((r = compute_slow(c))) return r;
    launch_rec_energy(c->ew, c->ew_sum, c->st, &c->launches);
    std::vector<double> h1;
    std::vector<float4> hf;
    if ((r = ddownload(c, h1, (const double *)c->ew_sum, 1)) || (r = ddownload(c, hf, (const float4 *)c->fslow, c->n))) return r;
    double s = h1[0] - kCoulomb * c->alpha / std::sqrt(3.14159265358979323846) * c->q2sum;
    for (const float4 &v : hf) s += (double)v.w;
    *e_slow = s;
    return poll_error(c);
}

extern "C" int jump_half(jump_ctx *c, double H_ps, int32_t with_accel, int64_t step) {
    if (!c) return JUMP_E_ARG;
    int r = ensure_f0(c);
    if (r) return r;
    r = run_update(c, ph_jump(c, H_ps, with_accel != 0, false, 1, 2, step), gr_f0(c), ph_none(), gr(nullptr), false);
    if (r) return r;
    return writeback(c);
}

// ---- life cycle ------------------------------------------------------------------------------------------
static int load_state(jump_ctx *c, const float *d_mass, const float *d_charge, const float *d_sigma, const float *d_eps) {
    launch_load(c->m, c->d_pos, c->d_vel, d_mass, d_charge, d_sigma, d_eps, c->kT, 0.5 * c->p.skin / c->w_norm, c->xs, c->vs, c->xl, c->lj, c->mi, c->hw, c->orig, c->st,
                &c->launches);
    CK(cudaGetLastError());
    return 0;
}

static int init_impl(jump_ctx *c, const jump_params *p, const float *d_mass, const float *d_charge, const float *d_sigma,
                     const float *d_eps, int n_bonds, const int32_t *d_bond_ij, const float *d_bond_k, const float *d_bond_r0,
                     int n_angles, const int32_t *d_angle_ijk, const float *d_angle_k, const float *d_angle_t0,
                     const int32_t *d_excl_ptr, const int32_t *d_excl_idx) {
    const int n = c->n = p->n_atoms;
    c->p = *p;
    c->kT = kKB * p->temperature_K;
    c->dt = p->dt_fs * 1e-3;
    c->alpha = p->ewald_alpha < 0.0 ? 3.8 / p->r_long : p->ewald_alpha;  // R-2
    c->lo = std::max(p->r_short - p->r_switch - p->skin, 0.0);
    c->rA = p->r_mid_in > 0.0 ? p->r_mid_in : p->r_short;   // R-10c: ring A = the switching zone by default
    c->rM = p->r_mid > 0.0 ? p->r_mid : c->rA;              // no outer split asked for: rings A and C
    if (c->rA > c->rM) c->rA = c->rM;
    double g1 = std::exp(-p->gamma_per_ps * c->dt);
    c->c1 = (float)g1;
    c->c2 = (float)std::sqrt(1.0 - g1 * g1);
    // host copies of the per-atom parameters (bounds) and the topology
    std::vector<float> hq, hs, he;
    int r;
    std::vector<float> hm;
    if ((r = ddownload(c, hq, d_charge, n)) || (r = ddownload(c, hs, d_sigma, n)) || (r = ddownload(c, he, d_eps, n)) ||
        (r = ddownload(c, hm, d_mass, n)))
        return r;
    {   // mass weights of the skin (R-10c): an atom may move w_i skin/2 between two list builds
        double sum = 0.0, mmin = 1e300;
        for (int i = 0; i < n; ++i) { if (!(hm[i] > 0.f)) return JUMP_E_ARG; sum += 1.0 / std::sqrt((double)hm[i]); mmin = std::min(mmin, (double)hm[i]); }
        c->w_norm = sum / n;
        c->w_max = (1.0 / std::sqrt(mmin)) / c->w_norm;
    }
    compute_bounds(c, hq, hs, he);
    // model constants
    Model &m = c->m;
    memset(&m, 0, sizeof m);
    m.n = n;
    for (int k = 0; k < 3; ++k) { m.box[k] = (float)p->box[k]; m.inv_box[k] = (float)(1.0 / p->box[k]); }
    m.rc = (float)p->r_short; m.h = (float)p->r_switch; m.inv_h = (float)(1.0 / p->r_switch);
    m.rlo = (float)(p->r_short - p->r_switch);
    m.rc2 = (float)(p->r_short * p->r_short); m.rlo2 = m.rlo * m.rlo;
    m.rlo2d = (p->r_short - p->r_switch) * (p->r_short - p->r_switch); m.rE2 = (float)(p->r_long * p->r_long);
    m.alpha = (float)c->alpha; m.alpha2 = (float)(c->alpha * c->alpha);
    m.beta = (float)(1.0 / c->kT);
    m.eps_jump = std::isinf(p->eps_jump) ? INFINITY : (float)p->eps_jump;
    m.eps_adaptive = p->eps_mode == 1 ? 1 : 0;
    m.combined = (p->flags & JUMP_F_COMBINED) ? 1 : 0;
    if (m.combined && (p->flags & (JUMP_F_COUL_JUMPS | JUMP_F_LJ_JUMPS)) != (JUMP_F_COUL_JUMPS | JUMP_F_LJ_JUMPS)) {
        c->err = "JUMP_F_COMBINED needs JUMP_F_COUL_JUMPS | JUMP_F_LJ_JUMPS (R-22)";
        return JUMP_E_ARG;
    }
    if (m.combined && m.eps_adaptive) {
        c->err = "JUMP_F_COMBINED with eps_mode 1 is not built (R-22 runs the constant-eps mechanism)";
        return JUMP_E_ARG;
    }
    {
        const double rlo = p->r_short - p->r_switch;
        const double eA = std::min(std::max(c->rA, rlo), p->r_long), eM = std::min(std::max(c->rM, eA), p->r_long);
        const double edge[4] = {rlo, eA, eM, p->r_long};
        for (int y = 0; y < 4; ++y) { m.ring2d[y] = edge[y] * edge[y]; m.ring2[y] = (float)m.ring2d[y]; }
        for (int y = 0; y < 3; ++y) {
            m.qmaxG[y] = (float)(c->qmax * c->G[y]);
            m.GV4se[y] = (float)(4.0 * std::sqrt(c->eps_max) * c->GV[y]);
        }
    }
    m.q_split = (float)(0.5 * (c->qmin_abs + c->qmax));
    m.half_skin2 = (float)(0.25 * p->skin * p->skin);
    m.hs = (float)(0.5 * p->skin);
    m.Wc = (float)(1.0 / (std::sqrt(c->kT * kKcal) * c->w_norm));
    m.w_max = (float)c->w_max;
    m.key0 = (unsigned)(p->seed & 0xffffffffu); m.key1 = (unsigned)(p->seed >> 32);
    // sort grid (R-10)
    SortGrid &g = c->g;
    double edge = p->cell_edge > 0.0 ? p->cell_edge : (p->r_long + p->skin * c->w_max) / 4.0;
    g.ncell = 1;
    for (int k = 0; k < 3; ++k) {
        g.gn[k] = std::max(1, (int)std::floor(p->box[k] / edge));
        g.scale[k] = (double)g.gn[k] / p->box[k];
        g.reach[k] = (int)std::ceil((p->r_long + p->skin * c->w_max) / (p->box[k] / g.gn[k]));
        if (g.reach[k] > 8 || g.gn[k] > 1023) return JUMP_E_ARG;  // stencil table of the row build (cell_edge too small); packed cells
        g.ncell *= g.gn[k];
    }
    // buffers
    if ((r = dalloc(c, &c->xs, n)) || (r = dalloc(c, &c->xs_nxt, n)) || (r = dalloc(c, &c->vs, n)) ||
        (r = dalloc(c, &c->vs_nxt, n)) || (r = dalloc(c, &c->xl, n)) || (r = dalloc(c, &c->xl_nxt, n)) || (r = dalloc(c, &c->x_build, n)) || (r = dalloc(c, &c->lj, n)) ||
        (r = dalloc(c, &c->lj_nxt, n)) || (r = dalloc(c, &c->mi, n)) || (r = dalloc(c, &c->mi_nxt, n)) || (r = dalloc(c, &c->hw, n)) || (r = dalloc(c, &c->hw_nxt, n)) ||
        (r = dalloc(c, &c->orig, n)) || (r = dalloc(c, &c->orig_nxt, n)) || (r = dalloc(c, &c->sorted_of, n)) || (r = dalloc(c, &c->cell_of, n)) ||
        (r = dalloc(c, &c->key, n)) || (r = dalloc(c, &c->tmp_orig, n)) || (r = dalloc(c, &c->tmp_src, n)) ||
        (r = dalloc(c, &c->cell_count, g.ncell + 1)) || (r = dalloc(c, &c->cell_fill, g.ncell + 1)) ||
        (r = dalloc(c, &c->cell_start, g.ncell + 1)) || (r = dalloc(c, &c->scan_sums, g.ncell / 4096 + 2)) ||
        (r = dalloc(c, &c->scan_offs, g.ncell / 4096 + 2)) || (r = dalloc(c, &c->fnb, n)) || (r = dalloc(c, &c->fbond, n)) ||
        (r = dalloc(c, &c->f0, n)) || (r = dalloc(c, &c->ftmp, n)) || (r = dalloc(c, &c->ftmp2, n)) ||
        (r = dalloc(c, &c->ke, n)) || (r = dalloc(c, &c->ctr, 1)))
        return r;
    CK(cudaMemsetAsync(c->ctr, 0, sizeof(Counters), c->st));
    CK(cudaMemsetAsync(c->fbond, 0, sizeof(float4) * n, c->st));   // atoms without bonded terms are never written
    {   // cell universe of ring C (R-10c): stencil of the cells within reach r_long + skin of a cell, in fp64 from the
        // caller's numbers (the oracle takes the same decisions from the same numbers)
        Universe &u = c->uni;
        memset(&u, 0, sizeof u);
        const double reach = p->r_long + p->skin * c->w_max;
        double w[3];
        for (int k = 0; k < 3; ++k) {
            w[k] = p->box[k] / g.gn[k];
            u.R[k] = (int)std::ceil(reach / w[k]);   // <= 8: checked above (g.reach)
            u.cnt[k] = std::min(2 * u.R[k] + 1, g.gn[k]);
        }
        u.nrow = u.cnt[2] * u.cnt[1];
        u.stride = (u.nrow + 1 + 7) / 8 * 8;
        u.inv_cnt1 = (65536 + u.cnt[1] - 1) / u.cnt[1];
        for (int a = 0; a < 17; ++a)
            for (int b = 0; b < 17; ++b) {
                const double gz = (a > 1 ? a - 1 : 0) * w[2], gy = (b > 1 ? b - 1 : 0) * w[1];
                const double rem = reach * reach - gz * gz - gy * gy;
                int v = -1;
                if (a <= u.R[2] && b <= u.R[1] && rem > 0.0) v = std::min(u.R[0], (int)std::floor(std::sqrt(rem) / w[0]) + 1);
                u.xr[a * 17 + b] = (signed char)v;
            }
        c->uni_cum = nullptr;
        if (coul_jumps(c) || lj_jumps(c)) {
            if ((r = dalloc(c, &c->uni_cum, (size_t)g.ncell * u.stride))) return r;
            CK(cudaMemsetAsync(c->uni_cum, 0, sizeof(unsigned short) * (size_t)g.ncell * u.stride, c->st));
        }
        u.cum = c->uni_cum;
        u.cell_of = c->cell_of;
    }
    c->event_cap = 0; c->events = nullptr;
    if (p->flags & JUMP_F_EVENT_LOG) {
        c->event_cap = std::min<long long>(std::max<long long>(1ll << 21, 512ll * n), 1ll << 25);
        if ((r = dalloc(c, &c->events, (size_t)c->event_cap))) return r;
    }
    // exclusions (own copy)
    c->excl_ptr = nullptr; c->excl_idx = nullptr;
    if (d_excl_ptr) {
        std::vector<int> hp;
        if ((r = ddownload(c, hp, (const int *)d_excl_ptr, n + 1))) return r;
        int tot = hp[n];
        if ((r = dalloc(c, &c->excl_ptr, n + 1)) || (r = dalloc(c, &c->excl_idx, tot))) return r;
        CK(cudaMemcpyAsync(c->excl_ptr, d_excl_ptr, sizeof(int) * (n + 1), cudaMemcpyDeviceToDevice, c->st));
        if (tot) CK(cudaMemcpyAsync(c->excl_idx, d_excl_idx, sizeof(int) * tot, cudaMemcpyDeviceToDevice, c->st));
    }
    // bonded terms as per-atom CSR over original indices
    {
        std::vector<int> hb, ha;
        std::vector<float> hbk, hbr, hak, hat;
        if ((r = ddownload(c, hb, (const int *)d_bond_ij, 2 * (size_t)n_bonds)) || (r = ddownload(c, hbk, d_bond_k, n_bonds)) ||
            (r = ddownload(c, hbr, d_bond_r0, n_bonds)) || (r = ddownload(c, ha, (const int *)d_angle_ijk, 3 * (size_t)n_angles)) ||
            (r = ddownload(c, hak, d_angle_k, n_angles)) || (r = ddownload(c, hat, d_angle_t0, n_angles)))
            return r;
        for (int v : hb) if (v < 0 || v >= n) return JUMP_E_ARG;
        for (int v : ha) if (v < 0 || v >= n) return JUMP_E_ARG;
        std::vector<int> bptr(n + 1, 0), aptr(n + 1, 0);
        for (int b = 0; b < n_bonds; ++b) { bptr[hb[2 * b] + 1]++; bptr[hb[2 * b + 1] + 1]++; }
        for (int a = 0; a < n_angles; ++a) for (int k = 0; k < 3; ++k) aptr[ha[3 * a + k] + 1]++;
        for (int i = 0; i < n; ++i) { bptr[i + 1] += bptr[i]; aptr[i + 1] += aptr[i]; }
        std::vector<int> bo(bptr[n]), bfill(bptr.begin(), bptr.end() - 1), ar(aptr[n]), aa(aptr[n]), ab(aptr[n]),
            afill(aptr.begin(), aptr.end() - 1);
        std::vector<float> bk(bptr[n]), br(bptr[n]), ak(aptr[n]), at(aptr[n]);
        for (int b = 0; b < n_bonds; ++b)
            for (int e = 0; e < 2; ++e) {
                int me = hb[2 * b + e], s = bfill[me]++;
                bo[s] = hb[2 * b + 1 - e]; bk[s] = hbk[b]; br[s] = hbr[b];
            }
        for (int a = 0; a < n_angles; ++a) {
            int i = ha[3 * a], j = ha[3 * a + 1], k = ha[3 * a + 2];  // j = vertex
            int s = afill[i]++; ar[s] = 0; aa[s] = j; ab[s] = k; ak[s] = hak[a]; at[s] = hat[a];
            s = afill[j]++;     ar[s] = 1; aa[s] = i; ab[s] = k; ak[s] = hak[a]; at[s] = hat[a];
            s = afill[k]++;     ar[s] = 2; aa[s] = j; ab[s] = i; ak[s] = hak[a]; at[s] = hat[a];
        }
        int *dbptr, *dbo, *daptr, *dar, *daa, *dab;
        float *dbk, *dbr, *dak, *dat;
        if ((r = dupload(c, &dbptr, bptr)) || (r = dupload(c, &dbo, bo)) || (r = dupload(c, &dbk, bk)) ||
            (r = dupload(c, &dbr, br)) || (r = dupload(c, &daptr, aptr)) || (r = dupload(c, &dar, ar)) ||
            (r = dupload(c, &daa, aa)) || (r = dupload(c, &dab, ab)) || (r = dupload(c, &dak, ak)) || (r = dupload(c, &dat, at)))
            return r;
        c->topo = Topo{dbptr, dbo, dbk, dbr, daptr, dar, daa, dab, dak, dat};
        // connected components of the bonded graph: those of at most three atoms become "small molecules" (one thread
        // each, every term evaluated once); the atoms of the others keep the per-atom CSR
        std::vector<int> root(n);
        for (int i = 0; i < n; ++i) root[i] = i;
        auto find = [&](int x) { while (root[x] != x) { root[x] = root[root[x]]; x = root[x]; } return x; };
        auto unite = [&](int x, int y) { x = find(x); y = find(y); if (x != y) root[std::max(x, y)] = std::min(x, y); };
        for (int b = 0; b < n_bonds; ++b) unite(hb[2 * b], hb[2 * b + 1]);
        for (int a = 0; a < n_angles; ++a) { unite(ha[3 * a], ha[3 * a + 1]); unite(ha[3 * a], ha[3 * a + 2]); }
        std::vector<int> csize(n, 0), cterms(n, 0), slot(n, -1);
        for (int i = 0; i < n; ++i) csize[find(i)]++;
        for (int b = 0; b < n_bonds; ++b) cterms[find(hb[2 * b])]++;
        for (int a = 0; a < n_angles; ++a) cterms[find(ha[3 * a])]++;
        std::vector<int4> mols;
        std::vector<MolType> mtypes;
        std::vector<int> big, mol_of(n, -1);
        for (int i = 0; i < n; ++i) {   // members of a component in ascending original index; root = smallest index
            const int r0 = find(i);
            if (cterms[r0] == 0) continue;   // no bonded term: the gradient stays zero
            if (csize[r0] > 3) { big.push_back(i); continue; }
            if (mol_of[r0] < 0) { mol_of[r0] = (int)mols.size(); mols.push_back(make_int4(-1, -1, -1, 0)); }
            int4 &mm = mols[mol_of[r0]];
            if (mm.x < 0) { mm.x = i; slot[i] = 0; } else if (mm.y < 0) { mm.y = i; slot[i] = 1; } else { mm.z = i; slot[i] = 2; }
        }
        std::vector<MolType> per_mol(mols.size());
        for (auto &t : per_mol) memset(&t, 0, sizeof t);
        bool fits = true;
        for (int b = 0; b < n_bonds && fits; ++b) {
            const int r0 = find(hb[2 * b]);
            if (csize[r0] > 3) continue;
            MolType &t = per_mol[mol_of[r0]];
            if (t.nb >= 3) { fits = false; break; }
            t.bp[t.nb] = slot[hb[2 * b]]; t.bq[t.nb] = slot[hb[2 * b + 1]]; t.bk[t.nb] = hbk[b]; t.br0[t.nb] = hbr[b]; t.nb++;
        }
        for (int a = 0; a < n_angles && fits; ++a) {
            const int r0 = find(ha[3 * a]);
            if (csize[r0] > 3) continue;
            MolType &t = per_mol[mol_of[r0]];
            if (t.na >= 3) { fits = false; break; }
            t.ai[t.na] = slot[ha[3 * a]]; t.av[t.na] = slot[ha[3 * a + 1]]; t.ak_[t.na] = slot[ha[3 * a + 2]];
            t.ak[t.na] = hak[a]; t.at0[t.na] = hat[a]; t.na++;
        }
        for (size_t q = 0; q < mols.size() && fits; ++q) {   // identical term tables share one type (a water box has one)
            int ty = -1;
            for (size_t u = 0; u < mtypes.size(); ++u) if (!memcmp(&mtypes[u], &per_mol[q], sizeof(MolType))) { ty = (int)u; break; }
            if (ty < 0) { if (mtypes.size() >= 64) { fits = false; break; } ty = (int)mtypes.size(); mtypes.push_back(per_mol[q]); }
            mols[q].w = ty;
        }
        if (!fits) {   // a small component with more terms than a type holds, or too many kinds: all atoms through the CSR
            big.clear();
            for (int i = 0; i < n; ++i) if (cterms[find(i)] > 0) big.push_back(i);
            mols.clear(); mtypes.clear();
        }
        int4 *dmols = nullptr; MolType *dtypes = nullptr; int *dbig = nullptr;
        if ((r = dupload(c, &dmols, mols)) || (r = dupload(c, &dtypes, mtypes)) || (r = dupload(c, &dbig, big))) return r;
        c->bonded = Bonded{(int)mols.size(), dmols, dtypes, (int)big.size(), dbig};
    }
    // rows: windows (R-10) and capacities from the mean density with head-room
    {
        const double vol = p->box[0] * p->box[1] * p->box[2], rho = n / vol, s = p->skin, rc = p->r_short, rE = p->r_long;
        int n_lj = 0;
        for (int i = 0; i < n; ++i) n_lj += he[i] > 0.f;
        const double rho_lj = n_lj / vol;
        // nominal windows [a, b) (R-10c); at a build the pair (i, j) is listed over [a - s_ij, b + s_ij), s_ij = (skin/2)(w_i + w_j)
        const double rlo = rc - p->r_switch;
        struct W { double a, b; int lj; } w[N_ROWS] = {
            {0.0, rc, 0},                 // S short list
            {rlo, c->rA, 0},              // A: candidates of ring [r_c-h, r_A)
            {c->rA, c->rM, 0},            // B: candidates of ring [r_A, r_M)
            {0.0, 0.0, 0},                // (unused)
            {0.0, rE, 0},                 // F: full list (lazy)
            {rc, rE, 1}};                 // W: LJ tail kept in F0 (R-13)
        const double smax = s * c->w_max;
        for (int k = 0; k < N_ROWS; ++k) {
            Row &R = c->rows[k];
            memset(&R, 0, sizeof R);
            const double hi = w[k].b + smax, lo = std::max(w[k].a - smax, 0.0);
            double expect = 4.0 / 3.0 * M_PI * std::max(hi * hi * hi - lo * lo * lo, 0.0) * (w[k].lj ? rho_lj : rho);
            R.cap = std::min(round32(1.6 * expect + 32.0), round32((double)n));
            R.lj_only = w[k].lj;
            R.ra = (float)w[k].a; R.rb = (float)w[k].b; R.ra_d = w[k].a; R.rb_d = w[k].b;
            R.lo_plus = k == ROW_W ? 1 : 0;
            R.r2max = (float)(hi * hi);
            c->row_active[k] = false;
            c->row_last_use[k] = 0;
        }
    }
    if ((r = load_state(c, d_mass, d_charge, d_sigma, d_eps))) return r;
    {   // the rows this mode reads on every step: active from the start, built with the first sort
        const bool jumps = coul_jumps(c) || lj_jumps(c);
        const bool want[N_ROWS] = {true, jumps, jumps, false, false, !lj_jumps(c)};
        for (int k = 0; k < N_ROWS; ++k)
            if (want[k]) { if ((r = alloc_row(c, k))) return r; c->row_active[k] = true; }
    }
    if ((r = resort_and_build(c, false))) return r;
    if ((r = compute_f0(c))) return r;
    if ((r = writeback(c))) return r;  // wrapped positions
    return poll_error(c);
}

extern "C" int jump_init(jump_ctx **out, const jump_params *p, float *d_pos, float *d_vel, const float *d_mass,
                         const float *d_charge, const float *d_lj_sigma, const float *d_lj_eps, int32_t n_bonds,
                         const int32_t *d_bond_ij, const float *d_bond_k, const float *d_bond_r0, int32_t n_angles,
                         const int32_t *d_angle_ijk, const float *d_angle_k, const float *d_angle_t0,
                         const int32_t *d_excl_ptr, const int32_t *d_excl_idx, void *cuda_stream) {
    if (!out || !p || !d_pos || !d_vel || !d_mass || !d_charge || !d_lj_sigma || !d_lj_eps) return JUMP_E_ARG;
    if (p->n_atoms <= 0 || n_bonds < 0 || n_angles < 0) return JUMP_E_ARG;
    if (p->n_inner <= 0 || (p->n_inner & 1)) return JUMP_E_ARG;
    if (!(p->r_switch > 0.0) || !(p->r_short > p->r_switch) || !(p->r_short < p->r_long)) return JUMP_E_ARG;
    for (int k = 0; k < 3; ++k) if (!(p->box[k] > 0.0) || p->r_long > 0.5 * p->box[k]) return JUMP_E_ARG;
    if ((p->eps_mode != 0 && p->eps_mode != 1) || (p->eps_mode == 1 && std::isinf(p->eps_jump)) || !(p->eps_jump > 0.0) || !(p->dt_fs > 0.0) || p->gamma_per_ps < 0.0 || !(p->temperature_K > 0.0))
        return JUMP_E_ARG;
    if (p->skin < 0.0 || p->nlist_every < 0) return JUMP_E_ARG;
    if (p->r_mid > 0.0 && (p->r_mid < p->r_short - p->r_switch || p->r_mid > p->r_long)) return JUMP_E_ARG;
    jump_ctx *c = new jump_ctx();
    c->st = (cudaStream_t)cuda_stream;
    c->st2 = nullptr; c->ev_fork = c->ev_join = nullptr; c->bonded_in_flight = false;
    if (cudaStreamCreateWithFlags(&c->st2, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        c->err = "side stream / events"; *out = c; return JUMP_E_CUDA;
    }
    c->d_pos = d_pos; c->d_vel = d_vel;
    c->step = c->outer = c->launches = 0;
    c->sticky = 0;
    c->pair_count = nullptr;
    c->moved_flag = nullptr;
    c->f0_valid = false;
    c->slow_valid = false;
    memset(&c->ew, 0, sizeof c->ew);
    c->vacf_v0 = nullptr; c->vacf_part = nullptr; c->msd_x0 = nullptr; c->msd_part = nullptr;
    c->fslow = nullptr; c->ew_sum = nullptr; c->q2sum = 0.0; c->outer1 = 0;
    c->prof = false;
    c->lanes = 0; c->uni_cum = nullptr; c->cell_of = nullptr;
    for (int k = 0; k < 4; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    int r = init_impl(c, p, d_mass, d_charge, d_lj_sigma, d_lj_eps, n_bonds, d_bond_ij, d_bond_k, d_bond_r0, n_angles,
                      d_angle_ijk, d_angle_k, d_angle_t0, d_excl_ptr, d_excl_idx);
    *out = c;  // returned even on failure so that jump_last_error can be read; free with jump_free
    return r;
}

extern "C" void jump_free(jump_ctx *c) {
    if (!c) return;
    prof_collect(c);
    if (c->st2) cudaStreamSynchronize(c->st2);
    for (auto &ev : c->prof_free) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->st2) cudaStreamDestroy(c->st2);
    for (void *q : c->owned) cudaFree(q);
    delete c;
}
extern "C" const char *jump_last_error(const jump_ctx *c) { return c ? c->err.c_str() : "null context"; }
extern "C" int64_t jump_get_step(const jump_ctx *c) { return c ? c->step : -1; }
extern "C" int64_t jump_get_launches(const jump_ctx *c) { return c ? c->launches : -1; }
extern "C" int jump_sync(jump_ctx *c) { return c ? poll_error(c) : JUMP_E_ARG; }

// ---- observers ---------------------------------------------------------------------------------------------
extern "C" int jump_get_forces(jump_ctx *c, int32_t which, float *d_out) {
    if (!c || !d_out) return JUMP_E_ARG;
    int r = 0;
    const float4 *src = nullptr;
    const float4 *src2 = nullptr;   // pieces are kept apart on the device (pair part + bonded part) and added on the way out
    switch (which) {
        case 0: r = compute_f0(c); src = c->fnb; src2 = c->fbond; break;
        case 1: r = compute_full(c, false); src = c->ftmp2; src2 = c->fbond; break;
        case 2: r = compute_long(c, c->ftmp); src = c->ftmp; break;
        case 3: r = bonded_only(c); src = c->fbond; break;
        case 4: r = compute_short_nb(c, c->fnb); src = c->fnb; break;
        case 5: c->slow_valid = false; r = compute_slow(c); src = c->fslow; break;
        default: return JUMP_E_ARG;
    }
    if (r) return r;
    launch_unsort3(c->n, src, src2, c->orig, d_out, c->st, &c->launches);
    CK(cudaGetLastError());
    return poll_error(c);
}

extern "C" int jump_get_energy(jump_ctx *c, double *e_kin, double *e_pot_full) {
    if (!c) return JUMP_E_ARG;
    int r;
    if (e_kin) {
        launch_kinetic(c->n, c->vs, c->mi, c->ke, c->st, &c->launches);
        std::vector<double> h;
        if ((r = ddownload(c, h, c->ke, c->n))) return r;
        double s = 0.0;
        for (double v : h) s += v;
        *e_kin = s;
    }
    if (e_pot_full) {
        if ((r = compute_full(c, true))) return r;
        std::vector<float4> h, hb;
        if ((r = ddownload(c, h, (const float4 *)c->ftmp2, c->n)) || (r = ddownload(c, hb, (const float4 *)c->fbond, c->n))) return r;
        double s = 0.0;
        for (int i = 0; i < c->n; ++i) s += (double)h[i].w + (double)hb[i].w;
        *e_pot_full = s;
    }
    return poll_error(c);
}

extern "C" int jump_get_stats(jump_ctx *c, jump_stats *o) {
    if (!c || !o) return JUMP_E_ARG;
    Counters h;
    CK(cudaMemcpyAsync(&h, c->ctr, sizeof h, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    memset(o, 0, sizeof *o);
    o->proposals = (int64_t)h.proposals; o->accepts = (int64_t)h.accepts; o->gt_attempts = (int64_t)h.gt_attempts;
    o->expiries = (int64_t)h.expiries; o->rebuilds = (int64_t)h.rebuilds;
    float f;
    memcpy(&f, &h.max_p_bits, 4); o->max_p = f;
    memcpy(&f, &h.max_gl_bits, 4); o->max_g_over_L = f;
    memcpy(&f, &h.max_disp2_bits, 4); o->max_disp = std::sqrt((double)f);
    for (int k = 0; k < N_ROWS; ++k) { o->max_row[k] = h.max_row[k]; o->cap_row[k] = c->rows[k].enabled ? c->rows[k].cap : 0; }
    poll_error(c);
    o->error = c->sticky;
    return 0;
}
extern "C" int jump_reset_stats(jump_ctx *c) {
    if (!c) return JUMP_E_ARG;
    Counters h;
    CK(cudaMemcpyAsync(&h, c->ctr, sizeof h, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    const unsigned long long ne = h.n_events;
    const unsigned nr = h.rebuilds;
    const int gs = h.go_step, lb = h.last_build;
    memset(&h, 0, sizeof h);
    h.n_events = ne; h.rebuilds = nr; h.go_step = gs; h.last_build = lb;
    CK(cudaMemcpyAsync(c->ctr, &h, sizeof h, cudaMemcpyHostToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));
    c->sticky = 0; c->err.clear();
    return 0;
}
extern "C" int jump_get_events(jump_ctx *c, jump_event *buf, int64_t cap, int64_t *n) {
    if (!c || !n) return JUMP_E_ARG;
    Counters h;
    CK(cudaMemcpyAsync(&h, c->ctr, sizeof h, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    *n = (int64_t)h.n_events;
    int64_t m = std::min<int64_t>(std::min<int64_t>(*n, cap), c->event_cap);
    if (buf && m > 0) {
        CK(cudaMemcpyAsync(buf, c->events, sizeof(jump_event) * m, cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
    }
    return 0;
}
extern "C" int jump_clear_events(jump_ctx *c) {
    if (!c) return JUMP_E_ARG;
    CK(cudaMemsetAsync(&c->ctr->n_events, 0, sizeof(unsigned long long), c->st));
    return 0;
}
extern "C" int jump_get_row(jump_ctx *c, int32_t which, int32_t atom, int32_t *host_out, int32_t cap) {
    if (!c || which < 0 || which >= N_ROWS || atom < 0 || atom >= c->n) return JUMP_E_ARG;
    int r;
    int i = 0, cnt = 0;
    CK(cudaMemcpyAsync(&i, c->sorted_of + atom, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    std::vector<int> row, orig;
    if (which == ROW_UNUSED) {   // the cell universe of the atom's home cell (ring C), through the lookup the chains use
        if (!c->uni_cum) return 0;
        int home = 0;
        unsigned short tot = 0;
        CK(cudaMemcpyAsync(&home, c->cell_of + i, sizeof(int), cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
        home &= 0x3fffffff;   // (bit 30: far-exclusion flag)
        const int hlin = ((home >> 20) * c->g.gn[1] + ((home >> 10) & 1023)) * c->g.gn[0] + (home & 1023);
        CK(cudaMemcpyAsync(&tot, c->uni_cum + (size_t)hlin * c->uni.stride + c->uni.nrow, sizeof tot, cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
        cnt = tot;
        int *d_list = nullptr;
        CK(cudaMalloc(&d_list, sizeof(int) * std::max(cnt, 1)));
        launch_universe_list(c->g, c->uni, c->cell_start, home, d_list, cnt, c->st, &c->launches);
        r = ddownload(c, row, (const int *)d_list, cnt);
        cudaFree(d_list);
        if (r) return r;
    } else {
        if ((r = need_row(c, which))) return r;
        const Row &R = c->rows[which];
        CK(cudaMemcpyAsync(&cnt, R.cnt + i, sizeof(int), cudaMemcpyDeviceToHost, c->st));
        CK(cudaStreamSynchronize(c->st));
        if ((r = ddownload(c, row, (const int *)(R.idx + (size_t)i * R.cap), cnt))) return r;
    }
    if ((r = ddownload(c, orig, (const int *)c->orig, c->n))) return r;
    for (int k = 0; k < cnt && k < cap; ++k) host_out[k] = orig[row[k] & 0x7fffffff];   // (bit 31: LJ flag of rows S, F, W)
    return cnt;
}
extern "C" int jump_get_images(jump_ctx *c, int32_t *d_img) {
    if (!c || !d_img) return JUMP_E_ARG;
    launch_images(c->n, c->xl, c->orig, d_img, c->st, &c->launches);
    CK(cudaGetLastError());
    return poll_error(c);
}
extern "C" int jump_rdf_accumulate(jump_ctx *c, int32_t lj_only, double r_max, int32_t n_bins, uint64_t *d_hist) {
    if (!c || !d_hist) return JUMP_E_ARG;
    // The cell table of the last sort indexes the sorted array, and an atom has moved by at most about the skin
    // since: the home cell of i is taken from its current position and the stencil reaches r_max + skin.
    if (launch_rdf(c->m, c->g, lj_only != 0, r_max, r_max + c->p.skin * c->w_max, n_bins, c->cell_start, c->xs, c->lj,
                   (unsigned long long *)d_hist, c->st, &c->launches))
        return JUMP_E_ARG;
    CK(cudaGetLastError());
    return 0;
}
extern "C" int jump_msd_mark(jump_ctx *c) {
    if (!c) return JUMP_E_ARG;
    int r;
    if (!c->msd_x0 && ((r = dalloc(c, &c->msd_x0, 3 * (size_t)c->n)) || (r = dalloc(c, &c->msd_part, (size_t)(c->n + 255) / 256 + 1)))) return r;
    launch_msd_mark(c->m, c->xs, c->xl, c->orig, c->msd_x0, c->st, &c->launches);
    CK(cudaGetLastError());
    return 0;
}
extern "C" int jump_msd(jump_ctx *c, int32_t lj_only, double *msd_out) {
    if (!c || !msd_out) return JUMP_E_ARG;
    if (!c->msd_x0) { c->err = "jump_msd_mark has not been called"; return JUMP_E_ARG; }
    const size_t nb = (size_t)(c->n + 255) / 256;
    launch_msd_sum(c->m, lj_only != 0, c->xs, c->xl, c->orig, c->lj, c->msd_x0, c->msd_part, c->msd_part + nb, c->st, &c->launches);
    CK(cudaGetLastError());
    std::vector<double2> h;
    int r = ddownload(c, h, (const double2 *)(c->msd_part + nb), 1);
    if (r) return r;
    *msd_out = h[0].y > 0.0 ? h[0].x / h[0].y : 0.0;
    return 0;
}
extern "C" int jump_vacf_mark(jump_ctx *c) {
    if (!c) return JUMP_E_ARG;
    int r;
    if (!c->vacf_v0 && ((r = dalloc(c, &c->vacf_v0, (size_t)c->n)) || (r = dalloc(c, &c->vacf_part, (size_t)(c->n + 255) / 256 + 1)))) return r;
    launch_vacf_mark(c->n, c->vs, c->orig, c->vacf_v0, c->st, &c->launches);
    CK(cudaGetLastError());
    return 0;
}
extern "C" int jump_vacf_dot(jump_ctx *c, int32_t lj_only, double *c_out) {
    if (!c || !c_out) return JUMP_E_ARG;
    if (!c->vacf_v0) { c->err = "jump_vacf_mark has not been called"; return JUMP_E_ARG; }
    const size_t nb = (size_t)(c->n + 255) / 256;
    launch_vacf_dot(c->n, lj_only != 0, c->vs, c->vacf_v0, c->orig, c->lj, c->vacf_part, c->vacf_part + nb, c->st, &c->launches);
    CK(cudaGetLastError());
    std::vector<double2> h;
    int r = ddownload(c, h, (const double2 *)(c->vacf_part + nb), 1);
    if (r) return r;
    *c_out = h[0].y > 0.0 ? h[0].x / h[0].y : 0.0;
    return 0;
}
extern "C" int jump_get_bounds(jump_ctx *c, double out[12]) {
    if (!c || !out) return JUMP_E_ARG;
    out[0] = c->G[0]; out[1] = c->G[1]; out[2] = c->GV[0]; out[3] = c->qmax;
    out[4] = c->eps_max; out[5] = c->sig_min; out[6] = c->sig_max; out[7] = c->rM;
    out[8] = c->G[2]; out[9] = c->GV[1]; out[10] = c->GV[2]; out[11] = c->rA;
    return 0;
}
extern "C" int jump_set_lax_skin(jump_ctx *c, int32_t on) {
    if (!c) return JUMP_E_ARG;
    if (on) c->p.flags |= JUMP_F_LAX_SKIN; else c->p.flags &= ~JUMP_F_LAX_SKIN;
    return 0;
}
extern "C" int jump_set_lanes(jump_ctx *c, int32_t lanes) {
    if (!c || !(lanes == 0 || lanes == 1 || lanes == 4 || lanes == 8 || lanes == 16)) return JUMP_E_ARG;
    c->lanes = lanes;
    return 0;
}
extern "C" int jump_refresh(jump_ctx *c) {
    if (!c) return JUMP_E_ARG;
    launch_reload(c->m, c->d_pos, c->d_vel, c->orig, c->xs, c->vs, c->xl, nullptr, nullptr, 0, c->mi, c->st, &c->launches);
    CK(cudaGetLastError());
    int r = resort_and_build(c, false);
    if (r) return r;
    if ((r = compute_f0(c))) return r;
    return poll_error(c);
}
extern "C" int jump_refresh_lazy(jump_ctx *c, int32_t *rebuilt) {
    if (!c) return JUMP_E_ARG;
    int r;
    if (!c->moved_flag && (r = dalloc(c, &c->moved_flag, 1))) return r;
    CK(cudaMemsetAsync(c->moved_flag, 0, sizeof(int), c->st));
    launch_reload(c->m, c->d_pos, c->d_vel, c->orig, c->xs, c->vs, c->xl, c->x_build, c->moved_flag, 1, c->mi, c->st, &c->launches);
    CK(cudaGetLastError());
    int moved = 0;
    CK(cudaMemcpyAsync(&moved, c->moved_flag, sizeof(int), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    c->slow_valid = false;
    if (moved && (r = resort_and_build(c, false))) return r;
    if (rebuilt) *rebuilt = moved;
    if ((r = compute_f0(c))) return r;
    return 0;
}

// ---- measurement helpers (bench.py) ------------------------------------------------------------------------
extern "C" int jump_set_profiling(jump_ctx *c, int32_t on) {
    if (!c) return JUMP_E_ARG;
    prof_collect(c);
    c->prof = on != 0;
    for (int k = 0; k < 4; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    return 0;
}
extern "C" int jump_get_profile(jump_ctx *c, double ms[4], int64_t count[4]) {
    if (!c || !ms || !count) return JUMP_E_ARG;
    prof_collect(c);
    for (int k = 0; k < 4; ++k) { ms[k] = c->prof_ms[k]; count[k] = c->prof_n[k]; }
    return 0;
}
extern "C" int jump_count_pairs(jump_ctx *c, int32_t which_row, double r_cut, int64_t *n_ordered) {
    if (!c || !n_ordered || which_row < 0 || which_row >= N_ROWS) return JUMP_E_ARG;
    int r = need_row(c, which_row);
    if (r) return r;
    if (!c->pair_count && (r = dalloc(c, &c->pair_count, 1))) return r;   // one counter, kept for the context's life
    unsigned long long *d = c->pair_count;
    CK(cudaMemsetAsync(d, 0, sizeof(unsigned long long), c->st));
    launch_count_pairs(c->m, c->rows[which_row], c->xs, (float)(r_cut * r_cut), d, c->st, &c->launches);
    unsigned long long h = 0;
    CK(cudaMemcpyAsync(&h, d, sizeof h, cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    *n_ordered = (int64_t)h;
    return 0;
}
