// sort_build.cu -- cell sort and row build (a2, a3).
//
// a1: atoms are binned on the "contract grid" of R-10 (cell edge >= (r_long+skin)/4) and stably sorted
//     by (cell key, original index): counting sort by cell + a per-cell sort by original index.
// a2/a3: one warp per atom walks the cells within reach in ascending key order and compacts the
//     atoms whose build-time minimum-image distance falls in each row's window [rmin, rmax) into
//     fixed-capacity rows.  Because the atom array is sorted by (cell key, original index), rows come
//     out in the canonical order of R-10 without any per-row sort (rows one can draw
//     from uniformly, with their counts N_M(i), N_L(i), N_V(i)).
#include "launch.h"

namespace jb {

__global__ void k_cell_key(int n, const float4 *__restrict__ xs, SortGrid g, int *__restrict__ key,
                           int *__restrict__ cell_count, Counters *ctr) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 x = xs[i];
    if (!(isfinite(x.x) && isfinite(x.y) && isfinite(x.z))) {
        atomicOr(&ctr->err, (unsigned)ERR_NAN);
        x.x = x.y = x.z = 0.f;
    }
    // the cell decision is taken in fp64 like the oracle's (R-10): floor(x * (gn / box)), clamped
    int cx = (int)floor((double)x.x * g.scale[0]);
    int cy = (int)floor((double)x.y * g.scale[1]);
    int cz = (int)floor((double)x.z * g.scale[2]);
    cx = min(max(cx, 0), g.gn[0] - 1);
    cy = min(max(cy, 0), g.gn[1] - 1);
    cz = min(max(cz, 0), g.gn[2] - 1);
    int k = (cz * g.gn[1] + cy) * g.gn[0] + cx;
    key[i] = k;
    atomicAdd(&cell_count[k], 1);
}

// exclusive scan of cell_count[0..ncell) into cell_start[0..ncell]; one block
__global__ void k_scan(int ncell, const int *__restrict__ cell_count, int *__restrict__ cell_start) {
    __shared__ int part[1024];
    int t = threadIdx.x, nt = blockDim.x;
    int per = (ncell + nt - 1) / nt;
    int lo = min(t * per, ncell), hi = min(lo + per, ncell);
    int s = 0;
    for (int k = lo; k < hi; ++k) s += cell_count[k];
    part[t] = s;
    __syncthreads();
    for (int off = 1; off < nt; off <<= 1) {
        int v = (t >= off) ? part[t - off] : 0;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    int run = part[t] - s;
    for (int k = lo; k < hi; ++k) {
        cell_start[k] = run;
        run += cell_count[k];
    }
    if (t == nt - 1) cell_start[ncell] = part[t];
}

__global__ void k_scatter(int n, const int *__restrict__ key, const int *__restrict__ orig,
                          const int *__restrict__ cell_start, int *__restrict__ cell_fill,
                          int *__restrict__ tmp_orig, int *__restrict__ tmp_src) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int k = key[i];
    int slot = cell_start[k] + atomicAdd(&cell_fill[k], 1);
    tmp_orig[slot] = orig[i];
    tmp_src[slot] = i;
}

// order each cell by original index (insertion sort; a cell holds a handful of atoms)
__global__ void k_cell_sort(int ncell, const int *__restrict__ cell_start, int *__restrict__ tmp_orig,
                            int *__restrict__ tmp_src) {
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    int lo = cell_start[c], hi = cell_start[c + 1];
    for (int a = lo + 1; a < hi; ++a) {
        int ko = tmp_orig[a], ks = tmp_src[a];
        int b = a - 1;
        while (b >= lo && tmp_orig[b] > ko) {
            tmp_orig[b + 1] = tmp_orig[b];
            tmp_src[b + 1] = tmp_src[b];
            --b;
        }
        tmp_orig[b + 1] = ko;
        tmp_src[b + 1] = ks;
    }
}

__global__ void k_permute(int n, const int *__restrict__ src, const int *__restrict__ new_orig,
                          const float4 *__restrict__ xs_in, const float4 *__restrict__ vs_in,
                          const float4 *__restrict__ xl_in, float4 *__restrict__ xl,
                          const float2 *__restrict__ lj_in, const float2 *__restrict__ mi_in,
                          float4 *__restrict__ xs, float4 *__restrict__ vs, float2 *__restrict__ lj,
                          float2 *__restrict__ mi, int *__restrict__ orig, int *__restrict__ sorted_of,
                          float4 *__restrict__ x_build) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s = src[i];
    float4 x = xs_in[s];
    xs[i] = x;
    x_build[i] = x;
    vs[i] = vs_in[s];
    xl[i] = xl_in[s];
    lj[i] = lj_in[s];
    mi[i] = mi_in[s];
    int o = new_orig[i];
    orig[i] = o;
    sorted_of[o] = i;
}

struct RowSet { Row r[N_ROWS]; };

// m-th value, in ascending order, of the cyclic cell range [start, start+cnt) mod gn
__device__ inline int cyc_val(int m, int start, int cnt, int gn) {
    int w = max(0, start + cnt - gn);
    return m < w ? m : start + m - w;
}
__device__ inline int cyc_off(int val, int c, int gn) {
    int o = val - c;
    if (2 * o > gn) o -= gn;
    else if (2 * o < -gn) o += gn;
    return o;
}

__global__ void __launch_bounds__(256) k_build_rows(Model m, SortGrid g, RowSet rows, float rmax_all,
                                                    const int *__restrict__ cell_start,
                                                    const float4 *__restrict__ xs, const float2 *__restrict__ lj,
                                                    const int *__restrict__ orig, const int *__restrict__ sorted_of,
                                                    const int *__restrict__ excl_ptr, const int *__restrict__ excl_idx,
                                                    Counters *ctr) {
    const unsigned full = 0xffffffffu;
    int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= m.n) return;
    const int i = warp;
    const float4 xi = xs[i];
    const bool lj_i = lj[i].y > 0.f;
    // my cell (same arithmetic as k_cell_key; x has not moved since)
    int c3[3];
    c3[0] = min(max((int)floor((double)xi.x * g.scale[0]), 0), g.gn[0] - 1);
    c3[1] = min(max((int)floor((double)xi.y * g.scale[1]), 0), g.gn[1] - 1);
    c3[2] = min(max((int)floor((double)xi.z * g.scale[2]), 0), g.gn[2] - 1);
    int start[3], cnt[3];
    float cs[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        cs[k] = m.box[k] / (float)g.gn[k];
        if (2 * g.reach[k] + 1 >= g.gn[k]) { start[k] = 0; cnt[k] = g.gn[k]; }
        else { start[k] = (c3[k] - g.reach[k] + g.gn[k]) % g.gn[k]; cnt[k] = 2 * g.reach[k] + 1; }
    }
    // exclusions of atom i (original indices -> sorted), first 32 kept in registers
    int ex_lo = 0, n_ex = 0;
    if (excl_ptr) { int o = orig[i]; ex_lo = excl_ptr[o]; n_ex = excl_ptr[o + 1] - ex_lo; }
    int ex_mine = (lane < n_ex) ? sorted_of[excl_idx[ex_lo + lane]] : -1;

    int count[N_ROWS];
#pragma unroll
    for (int k = 0; k < N_ROWS; ++k) count[k] = 0;
    const float rmax2 = rmax_all * rmax_all;
    const unsigned lt_mask = (1u << lane) - 1u;

    for (int mz = 0; mz < cnt[2]; ++mz) {
        int zc = cyc_val(mz, start[2], cnt[2], g.gn[2]);
        float dz = fmaxf(0.f, (float)(abs(cyc_off(zc, c3[2], g.gn[2])) - 1)) * cs[2];
        for (int my = 0; my < cnt[1]; ++my) {
            int yc = cyc_val(my, start[1], cnt[1], g.gn[1]);
            float dy = fmaxf(0.f, (float)(abs(cyc_off(yc, c3[1], g.gn[1])) - 1)) * cs[1];
            if (dz * dz + dy * dy >= rmax2) continue;
            int rowbase = (zc * g.gn[1] + yc) * g.gn[0];
            int w = max(0, start[0] + cnt[0] - g.gn[0]);
#pragma unroll 1
            for (int seg = 0; seg < 2; ++seg) {
                int ca = seg == 0 ? 0 : start[0], cb = seg == 0 ? w : start[0] + cnt[0] - w;
                if (cb <= ca) continue;
                int jb = cell_start[rowbase + ca], je = cell_start[rowbase + cb];
                for (int j0 = jb; j0 < je; j0 += 32) {
                    int j = j0 + lane;
                    bool valid = j < je && j != i;
                    float r2 = 0.f;
                    bool lj_j = false;
                    if (valid) {
                        float4 xj = xs[j];
                        float dx = min_image1(xi.x, xj.x, m.box[0], m.inv_box[0]);
                        float dy2 = min_image1(xi.y, xj.y, m.box[1], m.inv_box[1]);
                        float dz2 = min_image1(xi.z, xj.z, m.box[2], m.inv_box[2]);
                        r2 = dx * dx + dy2 * dy2 + dz2 * dz2;
                        if (lj_i) lj_j = lj[j].y > 0.f;
                    }
                    bool pass[N_ROWS];
                    bool any = false;
#pragma unroll
                    for (int k = 0; k < N_ROWS; ++k) {
                        const Row &R = rows.r[k];
                        pass[k] = R.enabled && valid && r2 >= R.r2min && r2 < R.r2max && (!R.lj_only || (lj_i && lj_j));
                        any |= pass[k];
                    }
                    if (n_ex > 0 && __any_sync(full, any)) {  // R-9: excluded pairs are never listed
                        bool ex = false;
                        for (int base = 0; base < n_ex; base += 32) {
                            int mine = ex_mine;
                            if (base > 0) mine = (base + lane < n_ex) ? sorted_of[excl_idx[ex_lo + base + lane]] : -1;
                            int lim = min(32, n_ex - base);
                            for (int e = 0; e < lim; ++e) ex |= (__shfl_sync(full, mine, e) == j);
                        }
                        if (ex) {
#pragma unroll
                            for (int k = 0; k < N_ROWS; ++k) pass[k] = false;
                        }
                    }
#pragma unroll
                    for (int k = 0; k < N_ROWS; ++k) {
                        const Row &R = rows.r[k];
                        if (!R.enabled) continue;
                        unsigned mask = __ballot_sync(full, pass[k]);
                        if (pass[k]) {
                            int pos = count[k] + __popc(mask & lt_mask);
                            if (pos < R.cap) R.idx[(size_t)i * R.cap + pos] = j;
                        }
                        count[k] += __popc(mask);
                    }
                }
            }
        }
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < N_ROWS; ++k) {
            const Row &R = rows.r[k];
            if (!R.enabled) continue;
            R.cnt[i] = min(count[k], R.cap);
            if (count[k] > R.cap) atomicOr(&ctr->err, (unsigned)ERR_OVERFLOW);
            if (count[k] > ctr->max_row[k]) atomicMax(&ctr->max_row[k], count[k]);
        }
    }
}

// ------------------------------------------------------------------------------------------
static inline int nblk(int n, int b) { return (n + b - 1) / b; }

void launch_sort(const SortArgs &a, cudaStream_t st, int64_t *launches) {
    const int B = 256;
    cudaMemsetAsync(a.cell_count, 0, sizeof(int) * (a.grid.ncell + 1), st);
    cudaMemsetAsync(a.cell_fill, 0, sizeof(int) * (a.grid.ncell + 1), st);
    k_cell_key<<<nblk(a.n, B), B, 0, st>>>(a.n, a.xs_in, a.grid, a.key, a.cell_count, a.ctr);
    k_scan<<<1, 1024, 0, st>>>(a.grid.ncell, a.cell_count, a.cell_start);
    k_scatter<<<nblk(a.n, B), B, 0, st>>>(a.n, a.key, a.orig_in, a.cell_start, a.cell_fill, a.tmp_orig, a.tmp_src);
    k_cell_sort<<<nblk(a.grid.ncell, B), B, 0, st>>>(a.grid.ncell, a.cell_start, a.tmp_orig, a.tmp_src);
    k_permute<<<nblk(a.n, B), B, 0, st>>>(a.n, a.tmp_src, a.tmp_orig, a.xs_in, a.vs_in, a.xl_in, a.xl, a.lj_in, a.mi_in, a.xs, a.vs,
                                          a.lj, a.mi, a.orig, a.sorted_of, a.x_build);
    *launches += 5;
}

void launch_build_rows(const Model &m, const SortGrid &g, const Row rows[N_ROWS], float rmax_all, const int *cell_start,
                       const float4 *xs, const float2 *lj, const int *orig, const int *sorted_of, const int *excl_ptr,
                       const int *excl_idx, Counters *ctr, cudaStream_t st, int64_t *launches) {
    RowSet rs;
    for (int k = 0; k < N_ROWS; ++k) rs.r[k] = rows[k];
    const int B = 256;
    long long threads = (long long)m.n * 32;
    k_build_rows<<<(unsigned)((threads + B - 1) / B), B, 0, st>>>(m, g, rs, rmax_all, cell_start, xs, lj, orig, sorted_of,
                                                                 excl_ptr, excl_idx, ctr);
    *launches += 1;
}

}  // namespace jb
