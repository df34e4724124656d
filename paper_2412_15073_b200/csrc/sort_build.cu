// sort_build.cu -- cell sort and row build (a2, a3).
//
// a1: atoms are binned on the "contract grid" of R-10 (cell edge >= (r_long+skin)/4) and stably sorted
//     by (cell key, original index): counting sort by cell + a per-cell sort by original index.
// a2/a3: one warp per atom walks the cells within reach in ascending key order and compacts the
//     atoms whose build-time minimum-image distance falls in each row's window [rmin, rmax) into
//     fixed-capacity rows.  Because the atom array is sorted by (cell key, original index), rows come
//     out in the canonical order of R-10 without any per-row sort (rows one can draw
//     from uniformly, with their counts N_M(i), N_L(i), N_V(i)).
#include <algorithm>
#include <cmath>
#include <type_traits>

#include <cooperative_groups.h>
#include "launch.h"

namespace jb {

// The per-element bodies of the sort passes (they are the passes of k_sort below).
__device__ __forceinline__ void cell_key_one(int i, const float4 *xs, const SortGrid &g, int *key, int *cell_count, Counters *ctr) {
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
// exclusive scan of cell_count[0..ncell) into cell_start[0..ncell]; one block (part: blockDim.x ints of shared memory)
__device__ __forceinline__ void scan_block(int ncell, const int *cell_count, int *cell_start, int *part) {
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
constexpr int SCAN_SLICE = 4096;   // cells per slice of the scan of large grids

__device__ __forceinline__ void scatter_one(int i, const int *key, const int *orig, const int *cell_start, int *cell_fill,
                                            int *tmp_orig, int *tmp_src) {
    int k = key[i];
    int slot = cell_start[k] + atomicAdd(&cell_fill[k], 1);
    tmp_orig[slot] = orig[i];
    tmp_src[slot] = i;
}
// order each cell by original index (insertion sort; a cell holds a handful of atoms)
__device__ __forceinline__ void cell_sort_one(int c, const int *cell_start, int *tmp_orig, int *tmp_src) {
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
struct RowSet { Row r[N_ROWS]; };

// d wrapped to the periodic image nearest to 0
__device__ inline float near_image1(float d, float L, float invL) {
    float t = d * invL + 12582912.f;   // round to nearest integer by the 1.5 * 2^23 trick
    t -= 12582912.f;
    return fmaf(-L, t, d);
}

// Shared-memory accesses of the filter loop through 32-bit shared-space addresses that the compiler must keep in
// registers (JB_KEEP makes a value opaque): left to itself, under the 72-register cap of 7 CTAs per SM, it
// recomputes lane, masks, the squared reach and the generic addresses of the tile and the queue in every iteration
// -- 18 of the loop's 47 instructions.
#define JB_KEEP(x) asm volatile("" : "+r"(x))
#define JB_KEEPF(x) asm volatile("" : "+f"(x))
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds128(unsigned a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ int lds32(unsigned a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void sts32(unsigned a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ int lds16(unsigned a) { unsigned short v; asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a) : "memory"); return (int)v; }
__device__ __forceinline__ void sts16(unsigned a, int v) { asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((unsigned short)v) : "memory"); }

// *p = v under a predicate, as ONE predicated store (the compiler's branch around a conditional store costs a
// convergence barrier pair and a jump per row and chunk in the row build's inner loop)
__device__ __forceinline__ void store_if(bool ok, int *p, int v) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %0, 0;\n\t@q st.global.s32 [%1], %2;\n\t}" ::"r"((int)ok), "l"(p), "r"(v) : "memory");
}

// Row build, one CTA per cell of the contract grid (per CX consecutive cells along x when the grid is large).
//  1. The candidate set of a cell is the same for all its atoms: the cells of a host-computed stencil (every cell
//     whose extent comes within rmax of this cell), visited in ascending cell key, i.e. a list of contiguous runs
//     [seg_beg, seg_beg + seg_len) of the sorted atom array.  The runs are found once per CTA, prefix-summed and
//     the candidates staged in shared memory in canonical order, BUILD_CHUNK at a time, ONCE for all atoms of the
//     cell.  A staged entry is (x, y, z | sorted index + LJ flag): in the FAST variant the coordinates are taken
//     relative to the cell centre and wrapped to the image nearest to it, so that the inner loop needs no minimum
//     image at all (valid when rmax + cell/2 <= box/2 in every dimension: then for every pair closer than rmax the
//     staged image IS the minimum image, and any other image is farther than rmax anyway).
//  2. Each warp takes the atoms a_beg + warp, + BUILD_WARPS, ... of the cell and scans the staged candidates 32 at
//     a time: distance, window tests of the selected rows, ballot compaction into the fixed-capacity rows (running
//     counts live in shared memory between chunks).  Exclusions and the atom itself are looked at only for
//     candidates closer than the atom's farthest excluded partner.
//  3. A candidate whose fp32 r^2 lies within BUILD_TIE of a window edge is decided again in fp64 from the full
//     positions x = xs + xl, with the oracle's expression d - L rint(d/L): membership at an edge is a discontinuous
//     decision (R-17) and the fp32 value of r^2 (error < 1e-3 A^2) would flip it where the fp64 oracle does not.
constexpr int BUILD_THREADS = 128;
constexpr int BUILD_WARPS = BUILD_THREADS / 32;
constexpr int BUILD_CX_MAX = 4;            // home cells per CTA (consecutive along x): 1 on small grids, more when the grid is large
constexpr int BUILD_CHUNK = 1024;           // candidates staged per pass
constexpr int BUILD_MAXSEG = 2 * 17 * 17;   // two x-runs per (z, y) cell row of the stencil
constexpr int BUILD_MAXATOMS = 32;          // atoms of a cell whose running counts are held at once
constexpr float BUILD_TIE = 4e-3f;          // A^2
constexpr float BUILD_TIE_R = 3e-4f;        // A: an fp32 distance this close to a window edge is re-decided in fp64

struct Stencil {
    int R[3];                 // cells on each side, per dimension
    signed char xr[17 * 17];  // [|oz| * 17 + |oy|] -> largest |ox| still within reach, -1: skip the (z, y) cell row
};

// MASK >= 0: bit k set = row k is built (compile-time row set of the common modes); MASK < 0: rows.r[k].enabled decides
template <int MASK, bool FAST>
__device__ __forceinline__ void build_rows_block(const Model &m, const SortGrid &g, const RowSet &rows, const Stencil &stn, float rmax_all,
                                                 int CX, const int *__restrict__ cell_start, const float4 *__restrict__ xs,
                                                 const float4 *__restrict__ xl, const float2 *__restrict__ lj,
                                                 const float2 *__restrict__ hw, const int *__restrict__ orig,
                                                 const int *__restrict__ sorted_of, const int *__restrict__ excl_ptr,
                                                 const int *__restrict__ excl_idx, Counters *ctr, int *__restrict__ cell_of,
                                                 float far2, const int bid) {
    __shared__ int seg_beg[BUILD_MAXSEG];       // stencil runs in ascending cell key (many are empty) ...
    __shared__ int seg_pre[BUILD_MAXSEG + 1];   // ... their lengths, then (length << 10 | non-empty) prefix sums
    __shared__ int run_beg[BUILD_MAXSEG];       // the non-empty runs, compacted: first atom ...
    __shared__ int run_pre[BUILD_MAXSEG + 1];   // ... and exclusive prefix of the lengths
    __shared__ float4 tile[BUILD_CHUNK];        // (x, y, z, sorted index | LJ flag in bit 31)
    __shared__ float tile_w[BUILD_CHUNK];       // (skin/2) w_j: the candidate's share of the pair's skin (R-10c)
    __shared__ int scan_tmp[BUILD_THREADS];
    __shared__ int s_count[BUILD_MAXATOMS][N_ROWS];
    __shared__ unsigned short s_queue[BUILD_WARPS][128];   // per warp: slots of the candidates that passed the distance filter
    const unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // the CTA's home: CX consecutive cells along x (their atoms are contiguous in the sorted array)
    const int nbx = (g.gn[0] + CX - 1) / CX;
    int c3[3];
    c3[0] = (bid % nbx) * CX;
    c3[1] = (bid / nbx) % g.gn[1];
    c3[2] = bid / (nbx * g.gn[1]);
    const int ncx = min(CX, g.gn[0] - c3[0]);
    const int cell0 = (c3[2] * g.gn[1] + c3[1]) * g.gn[0] + c3[0];
    const int a_beg = cell_start[cell0], a_end = cell_start[cell0 + ncx];
    if (a_end == a_beg) return;
    float ctr3[3];   // centre of the home cells (FAST: origin of the staged coordinates)
    int start[3], cnt[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        ctr3[k] = ((float)c3[k] + (k == 0 ? 0.5f * (float)ncx : 0.5f)) * (m.box[k] / (float)g.gn[k]);
        if (2 * stn.R[k] + 1 >= g.gn[k]) { start[k] = 0; cnt[k] = g.gn[k]; }
        else { start[k] = (c3[k] - stn.R[k] + g.gn[k]) % g.gn[k]; cnt[k] = 2 * stn.R[k] + 1; }
    }
    // ---- 1. runs of the stencil in ascending cell key -------------------------------------------------------
    const int nzy = cnt[2] * cnt[1], nseg = 2 * nzy;
    for (int p = tid; p < nzy; p += BUILD_THREADS) {
        int mz = p / cnt[1], my = p - mz * cnt[1];
        int zc = cyc_val(mz, start[2], cnt[2], g.gn[2]), yc = cyc_val(my, start[1], cnt[1], g.gn[1]);
        int oz = abs(cyc_off(zc, c3[2], g.gn[2])), oy = abs(cyc_off(yc, c3[1], g.gn[1]));
        int xm = stn.xr[oz * 17 + oy];
        int b0 = 0, n0 = 0, b1 = 0, n1 = 0;
        if (xm >= 0) {
            int rowbase = (zc * g.gn[1] + yc) * g.gn[0];
            if (2 * xm + ncx >= g.gn[0]) {
                b0 = cell_start[rowbase]; n0 = cell_start[rowbase + g.gn[0]] - b0;
            } else {
                int xs0 = (c3[0] - xm + g.gn[0]) % g.gn[0], xc = 2 * xm + ncx;
                int w = max(0, xs0 + xc - g.gn[0]);          // cells wrapped to the low end come first
                if (w > 0) { b0 = cell_start[rowbase]; n0 = cell_start[rowbase + w] - b0; }
                b1 = cell_start[rowbase + xs0]; n1 = cell_start[rowbase + xs0 + xc - w] - b1;
            }
        }
        seg_beg[2 * p] = b0; seg_pre[2 * p + 1] = n0;
        seg_beg[2 * p + 1] = b1; seg_pre[2 * p + 2] = n1;
    }
    if (tid == 0) seg_pre[0] = 0;
    __syncthreads();
    {   // inclusive scan of (length << 10 | non-empty) over seg_pre[1..nseg] (each thread a contiguous slice, then a
        // block scan of the slice sums): one pass gives the candidate offsets and the compacted run indices
        int per = (nseg + BUILD_THREADS - 1) / BUILD_THREADS;
        int lo = min(tid * per, nseg), hi = min(lo + per, nseg);
        int sum = 0;
        for (int k = lo; k < hi; ++k) { int len = seg_pre[k + 1]; sum += (len << 10) | (len > 0 ? 1 : 0); }
        scan_tmp[tid] = sum;
        __syncthreads();
        for (int off = 1; off < BUILD_THREADS; off <<= 1) {
            int v = tid >= off ? scan_tmp[tid - off] : 0;
            __syncthreads();
            scan_tmp[tid] += v;
            __syncthreads();
        }
        int run = scan_tmp[tid] - sum;
        for (int k = lo; k < hi; ++k) {
            int len = seg_pre[k + 1];
            if (len > 0) { run_beg[run & 1023] = seg_beg[k]; run_pre[run & 1023] = run >> 10; }
            run += (len << 10) | (len > 0 ? 1 : 0);
        }
        if (tid == BUILD_THREADS - 1) { seg_pre[0] = run; run_pre[run & 1023] = run >> 10; }
    }
    __syncthreads();
    const int total = seg_pre[0] >> 10, nrun = seg_pre[0] & 1023;
    const float rmax2t = rmax_all * rmax_all + BUILD_TIE;
    const unsigned lt_mask = (1u << lane) - 1u;
#define JB_ROW_ON(k) (MASK >= 0 ? (((MASK) >> (k)) & 1) != 0 : rows.r[k].enabled != 0)
    // window constants of the rows, read once (the compile-time row sets also know which rows have a lower edge: A, B, W;
    // and that only W counts it from r - s_ij)
#define JB_HAS_LO(k) (MASK >= 0 ? ((k) == ROW_A || (k) == ROW_B || (k) == ROW_W) : e_lo[k] > 0.f)
#define JB_LO_PLUS(k) (MASK >= 0 ? (k) == ROW_W : rows.r[k].lo_plus != 0)
    float e_hi[N_ROWS], e_lo[N_ROWS];
    int e_cap[N_ROWS];
#pragma unroll
    for (int k = 0; k < N_ROWS; ++k) {
        e_hi[k] = JB_ROW_ON(k) ? rows.r[k].rb : 0.f;
        e_lo[k] = JB_ROW_ON(k) ? rows.r[k].ra : 0.f;
        e_cap[k] = JB_ROW_ON(k) ? rows.r[k].cap : 0;
    }
    unsigned tile_a = smem_u32(tile) + 16u * (unsigned)lane;   // this lane's column of the staged chunk
    unsigned que_a = smem_u32(s_queue[warp]);
    unsigned lt_keep = lt_mask;
    float reach2 = rmax2t;
    int lane_keep = lane;
    unsigned tilew_a = smem_u32(tile_w);
    JB_KEEP(tile_a); JB_KEEP(que_a); JB_KEEP(lt_keep); JB_KEEPF(reach2); JB_KEEP(lane_keep); JB_KEEP(tilew_a);
    for (int g0 = a_beg; g0 < a_end; g0 += BUILD_MAXATOMS) {   // one pass unless a cell holds > BUILD_MAXATOMS atoms
        const int g1 = min(g0 + BUILD_MAXATOMS, a_end);
        for (int t = tid; t < BUILD_MAXATOMS * N_ROWS; t += BUILD_THREADS) (&s_count[0][0])[t] = 0;
        for (int c0 = 0; c0 < total || c0 == 0; c0 += BUILD_CHUNK) {
            const int c1 = min(c0 + BUILD_CHUNK, total);
            const int npad = (c1 - c0 + 63) & ~63;   // (the filter takes two groups of 32 per iteration)
            __syncthreads();   // the previous chunk has been consumed (and s_count is zeroed)
            {   // ---- stage [c0, c1): each warp takes a contiguous quarter of the chunk, 32 consecutive candidates per
                // iteration (coalesced loads); a lane's run is found by one bisection and then advanced linearly --
                // by about one run per iteration, since consecutive iterations of a lane are 32 candidates apart
                constexpr int PER_WARP = BUILD_CHUNK / BUILD_WARPS;
                int q = c0 + warp * PER_WARP + lane, r = 0;
                const int q_end = min(c0 + (warp + 1) * PER_WARP, c1);
                if (q < q_end) {
                    int hi_r = nrun - 1;   // last run with run_pre[r] <= q
                    while (r < hi_r) { int mid = (r + hi_r + 1) >> 1; if (run_pre[mid] <= q) r = mid; else hi_r = mid - 1; }
                }
                for (; q < q_end; q += 32) {
                    while (run_pre[r + 1] <= q) ++r;
                    const int j = run_beg[r] + (q - run_pre[r]);
                    float4 x = xs[j];
                    if (FAST) {
                        x.x = near_image1(x.x - ctr3[0], m.box[0], m.inv_box[0]);
                        x.y = near_image1(x.y - ctr3[1], m.box[1], m.inv_box[1]);
                        x.z = near_image1(x.z - ctr3[2], m.box[2], m.inv_box[2]);
                    }
                    x.w = __int_as_float(j | (lj[j].y > 0.f ? (int)0x80000000 : 0));
                    tile[q - c0] = x;
                    tile_w[q - c0] = hw[j].x;
                }
                for (int q = (c1 - c0) + tid; q < npad; q += BUILD_THREADS) { tile[q] = make_float4(nanf(""), 0.f, 0.f, 0.f); tile_w[q] = 0.f; }   // padding: r^2 = NaN fails every test
            }
            __syncthreads();
            // ---- 2./3. the atoms of the cell against the staged chunk ---------------------------------------------
            for (int i = g0 + warp; i < g1; i += BUILD_WARPS) {
                const float4 xi4 = xs[i];
                float xi = xi4.x, yi = xi4.y, zi = xi4.z;
                if (FAST) {
                    xi = near_image1(xi - ctr3[0], m.box[0], m.inv_box[0]);
                    yi = near_image1(yi - ctr3[1], m.box[1], m.inv_box[1]);
                    zi = near_image1(zi - ctr3[2], m.box[2], m.inv_box[2]);
                }
                JB_KEEPF(xi); JB_KEEPF(yi); JB_KEEPF(zi);   // (else recomputed from xs[i] in every iteration of the scan)
                const bool lj_i = lj[i].y > 0.f;
                const float2 hw_i = hw[i];
                const float hsw_i = hw_i.x;   // (skin/2) w_i
                // excluded partners (R-9): the first four in every lane, and the largest distance to any of them
                int ex_lo = 0, n_ex = 0;
                if (excl_ptr) { int o = orig[i]; ex_lo = excl_ptr[o]; n_ex = excl_ptr[o + 1] - ex_lo; }
                float exr2 = 0.f;
                int ex_mine = -1;
                for (int base = 0; base < n_ex; base += 32) {
                    int p = (base + lane < n_ex) ? sorted_of[excl_idx[ex_lo + base + lane]] : -1;
                    if (base == 0) ex_mine = p;
                    if (p >= 0) {
                        float4 xp = xs[p];
                        float ddx = min_image1(xi4.x, xp.x, m.box[0], m.inv_box[0]);
                        float ddy = min_image1(xi4.y, xp.y, m.box[1], m.inv_box[1]);
                        float ddz = min_image1(xi4.z, xp.z, m.box[2], m.inv_box[2]);
                        exr2 = fmaxf(exr2, ddx * ddx + ddy * ddy + ddz * ddz);
                    }
                }
                exr2 = __uint_as_float(__reduce_max_sync(full, __float_as_uint(exr2)));   // non-negative floats order as uints
                // an excluded partner that could be found in jump ring C (R-10c): the chains then check the universe's
                // candidates against the exclusion list (never so in water)
                if (cell_of && lane == 0 && c0 == 0 && exr2 > far2) cell_of[i] |= 1 << 30;
                exr2 = exr2 * 1.0001f + 2e-3f;   // also catches the atom itself (r^2 = 0)
                int ex4[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) ex4[e] = __shfl_sync(full, ex_mine, e);
                int count[N_ROWS];
                int *rbase[N_ROWS];
#pragma unroll
                for (int k = 0; k < N_ROWS; ++k) {
                    count[k] = JB_ROW_ON(k) ? s_count[i - g0][k] : 0;
                    rbase[k] = JB_ROW_ON(k) ? rows.r[k].idx + (size_t)i * rows.r[k].cap : nullptr;
                }
                // The scan is instantiated twice: an atom without LJ (two thirds of a water box) has no W row, and
                // its copy of the loop carries no test, ballot or counter for them (MASK >= 0; a branch on this
                // inside the unrolled row loop was measured slower than the work it skips).
                auto scan = [&](auto lj_tag) {
                    constexpr bool LJ_I = decltype(lj_tag)::value;
#define JB_ROW_SCAN(k) (JB_ROW_ON(k) && (LJ_I || MASK < 0 || (k) != ROW_W))
#define JB_LJ_ROW(k) (MASK >= 0 ? (k) == ROW_W : rows.r[k].lj_only != 0)   // W is the LJ-only row
                    // Two passes per 32 candidates.  Filter: distance only; the slots of the candidates within reach
                    // of the largest window go, in order, to a 64-entry ring buffer of the warp.  Windows: whenever 32
                    // are waiting they are taken off the buffer, one per lane -- every lane of the expensive part
                    // (window tests, ties, ballot compaction) then carries a candidate that can be listed, where
                    // the chunk itself has them in 4 lanes out of 10.  The buffer keeps the candidates' order, and so
                    // do the rows.
                    int q_head = 0, q_n = 0;
                    auto dist2 = [&](const float4 &xj) {
                        float dx, dy, dz;
                        if (FAST) { dx = xi - xj.x; dy = yi - xj.y; dz = zi - xj.z; }
                        else {
                            dx = min_image1(xi, xj.x, m.box[0], m.inv_box[0]);
                            dy = min_image1(yi, xj.y, m.box[1], m.inv_box[1]);
                            dz = min_image1(zi, xj.z, m.box[2], m.inv_box[2]);
                        }
                        return dx * dx + dy * dy + dz * dz;
                    };
                    auto windows = [&](const int n_live) {
                        __syncwarp();
                        const int slot = lane_keep < n_live ? lds16(que_a + 2u * (unsigned)((q_head + lane_keep) & 127)) : 0;
                        const float4 xj = lds128(tile_a + 16u * (unsigned)(slot - lane_keep));
                        const int jraw = __float_as_int(xj.w);
                        const int j = jraw & 0x7fffffff;
                        const float r2 = dist2(xj);
                        bool valid = lane_keep < n_live;
                        const bool nearby = valid && r2 <= exr2;
                        if (__any_sync(full, nearby)) {   // the atom itself and excluded pairs are never listed (R-9)
                            bool ex = (j == i) | (j == ex4[0]) | (j == ex4[1]) | (j == ex4[2]) | (j == ex4[3]);
                            if (n_ex > 4) {
                                for (int base = 0; base < n_ex; base += 32) {
                                    int mine = (base + lane < n_ex) ? sorted_of[excl_idx[ex_lo + base + lane]] : -1;
                                    int lim = min(32, n_ex - base);
                                    for (int e = 0; e < lim; ++e) ex |= (__shfl_sync(full, mine, e) == j);
                                }
                            }
                            valid = valid && !ex;
                        }
                        const bool ljp = LJ_I && jraw < 0;
                        // window of this pair in row k: [ra - s_ij, rb + s_ij), s_ij = (skin/2)(w_i + w_j) (row W: from ra + s_ij),
                        // tested on r -/+ s_ij against the row's constants
                        const float sij = hsw_i + __int_as_float(lds32(tilew_a + 4u * (unsigned)slot));
                        const float r = r2 * rsqrt_fast(fmaxf(r2, 1e-12f));
                        const float rm = r - sij, rp = r + sij;
                        bool pass[N_ROWS];
                        float edge_gap = 1e30f;   // distance of r to the nearest window edge of a scanned row
#pragma unroll
                        for (int k = 0; k < N_ROWS; ++k) {
                            pass[k] = false;
                            if (!JB_ROW_SCAN(k)) continue;
                            bool in = rm < e_hi[k];
                            edge_gap = fminf(edge_gap, fabsf(rm - e_hi[k]));
                            if (JB_HAS_LO(k)) {
                                const float t = JB_LO_PLUS(k) ? rm : rp;
                                in = in && t >= e_lo[k];
                                edge_gap = fminf(edge_gap, fabsf(t - e_lo[k]));
                            }
                            pass[k] = valid && (!JB_LJ_ROW(k) || ljp) && in;
                        }
                        const bool tie = valid && edge_gap < BUILD_TIE_R;
                        if (tie) {   // decide in fp64 from the full positions, like the oracle
                            float4 hi_j = xs[j], li = xl[i], lo_j = xl[j];
                            double d[3] = {((double)xi4.x + (double)li.x) - ((double)hi_j.x + (double)lo_j.x),
                                           ((double)xi4.y + (double)li.y) - ((double)hi_j.y + (double)lo_j.y),
                                           ((double)xi4.z + (double)li.z) - ((double)hi_j.z + (double)lo_j.z)};
                            double r2d = 0.0;
#pragma unroll
                            for (int k = 0; k < 3; ++k) {
                                double L = (double)m.box[k];
                                d[k] -= L * rint(d[k] / L);
                                r2d += d[k] * d[k];
                            }
                            const float2 hw_j = hw[j];
                            const double sd = ((double)hw_i.x + (double)hw_i.y) + ((double)hw_j.x + (double)hw_j.y);   // s_ij in fp64
#pragma unroll
                            for (int k = 0; k < N_ROWS; ++k) {
                                if (!JB_ROW_SCAN(k)) continue;
                                const Row &R = rows.r[k];
                                const double hi = R.rb_d + sd;
                                const double lo = R.ra > 0.f ? (R.lo_plus ? R.ra_d + sd : fmax(R.ra_d - sd, 0.0)) : 0.0;
                                pass[k] = (!JB_LJ_ROW(k) || ljp) && r2d >= lo * lo && r2d < hi * hi;
                            }
                        }
#pragma unroll
                        for (int k = 0; k < N_ROWS; ++k) {
                            if (!JB_ROW_SCAN(k)) continue;
                            const unsigned mask = __ballot_sync(full, pass[k]);
                            const int pos = count[k] + __popc(mask & lt_mask);
                            // rows the pair kernel reads carry j's LJ flag in bit 31; the jump rows A, B plain indices
                            store_if(pass[k] && pos < e_cap[k], rbase[k] + pos, (k == ROW_A || k == ROW_B) ? j : jraw);
                            count[k] += __popc(mask);
                        }
                        __syncwarp();   // the slots just read may be written again
                    };
                    for (int q0 = 0; q0 < npad; q0 += 64) {   // two groups of 32 per iteration: half the loop and vote overhead
                        const bool in_a = dist2(lds128(tile_a + 16u * (unsigned)q0)) < reach2;   // false for the NaN of a padding entry
                        const bool in_b = dist2(lds128(tile_a + 16u * (unsigned)(q0 + 32))) < reach2;
                        const unsigned ma = __ballot_sync(full, in_a), mb = __ballot_sync(full, in_b);
                        if ((ma | mb) == 0u) continue;
                        const int at = q_head + q_n;
                        if (in_a) sts16(que_a + 2u * (unsigned)((at + __popc(ma & lt_keep)) & 127), q0 + lane_keep);
                        if (in_b) sts16(que_a + 2u * (unsigned)((at + __popc(ma) + __popc(mb & lt_keep)) & 127), q0 + 32 + lane_keep);
                        q_n += __popc(ma) + __popc(mb);   // at most 31 + 64 of the 128 entries
                        while (q_n >= 32) { windows(32); q_head = (q_head + 32) & 127; q_n -= 32; }
                    }
                    if (q_n > 0) windows(q_n);
#undef JB_ROW_SCAN
#undef JB_LJ_ROW
                };
                if (lj_i) scan(std::true_type{}); else scan(std::false_type{});
                if (c1 >= total) {   // last chunk: publish the counts
                    if (lane == 0) {
#pragma unroll
                        for (int k = 0; k < N_ROWS; ++k) {
                            if (!JB_ROW_ON(k)) continue;
                            const Row &R = rows.r[k];
                            R.cnt[i] = min(count[k], R.cap);
                            if (count[k] > R.cap) atomicOr(&ctr->err, (unsigned)ERR_OVERFLOW);
                            if (count[k] > ctr->max_row[k]) atomicMax(&ctr->max_row[k], count[k]);
                        }
                    }
                } else if (lane == 0) {
#pragma unroll
                    for (int k = 0; k < N_ROWS; ++k) if (JB_ROW_ON(k)) s_count[i - g0][k] = count[k];
                }
            }
        }
        __syncthreads();   // before s_count is zeroed for the next group of atoms
    }
#undef JB_ROW_ON
#undef JB_HAS_LO
#undef JB_LO_PLUS
}

// resident grid over the nblocks home-cell groups (work queue 0 of the counters)
template <int MASK, bool FAST>
__global__ void __launch_bounds__(BUILD_THREADS, 7) k_build_rows(Model m, SortGrid g, RowSet rows, Stencil stn, float rmax_all, int CX,
                                                              const int *__restrict__ cell_start,
                                                              const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                              const float2 *__restrict__ lj, const float2 *__restrict__ hw,
                                                              const int *__restrict__ orig, const int *__restrict__ sorted_of,
                                                              const int *__restrict__ excl_ptr, const int *__restrict__ excl_idx,
                                                              Counters *ctr, int *__restrict__ cell_of, float far2,
                                                              const int *__restrict__ go, int want, int nblocks) {
    if (go && *go != want) return;
    __shared__ int s_item;
    for (;;) {
        const int bid = work_fetch(ctr, 0, &s_item);
        if (bid >= nblocks) break;
        build_rows_block<MASK, FAST>(m, g, rows, stn, rmax_all, CX, cell_start, xs, xl, lj, hw, orig, sorted_of, excl_ptr, excl_idx,
                                     ctr, cell_of, far2, bid);
    }
    work_leave(ctr, 0);
}

// ---- cell universe of jump ring C (R-10c) -----------------------------------------------------------------------
// One warp per home cell: the lengths of its stencil rows (two cell_start differences each), prefix-summed into
// cum[h][0 .. nrow]; cum[h][nrow] is the size of the universe, N_C of every atom of the cell.
__device__ __forceinline__ void universe_cell(const SortGrid &g, const Universe &u, const int *cell_start, unsigned short *cum,
                                              Counters *ctr, int h, int lane) {
    if (cell_start[h + 1] == cell_start[h]) return;   // no atom lives here: the row is never read
    const int cx = h % g.gn[0], cy = (h / g.gn[0]) % g.gn[1], cz = h / (g.gn[0] * g.gn[1]);
    unsigned short *out = cum + (size_t)h * u.stride;
    int run = 0;
    for (int p0 = 0; p0 < u.nrow; p0 += 32) {
        const int p = p0 + lane;
        int len = 0;
        if (p < u.nrow) {
            int b0, n0, b1, n1;
            const int mz = p / u.cnt[1];
            universe_row(g, u, cell_start, cx, cy, cz, mz, p - mz * u.cnt[1], b0, n0, b1, n1);
            len = n0 + n1;
        }
        int inc = len;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int up = __shfl_up_sync(0xffffffffu, inc, off);
            if (lane >= off) inc += up;
        }
        if (p < u.nrow) out[p] = (unsigned short)min(run + inc - len, 65535);
        run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) {
        out[u.nrow] = (unsigned short)min(run, 65535);
        if (run >= 65535) atomicOr(&ctr->err, (unsigned)ERR_OVERFLOW);   // 16-bit running sums
    }
}
__global__ void k_universe_list(SortGrid g, Universe u, const int *__restrict__ cell_start, int h, int n, int *__restrict__ out) {   // h: packed home cell
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = universe_pick(g, u, cell_start, h, k);
}

// ------------------------------------------------------------------------------------------
// The whole sort in ONE cooperative launch: zero the counts, keys, scan, scatter, per-cell order, permute into scratch,
// copy back (whether a conditional sort ran is known on the device only: no pointer swap), the running sums of the cell
// universe -- with grid-wide barriers between the passes.  The list kernels are enqueued at every step to return at once
// on most of them: one idle launch instead of eleven (two memsets and nine kernels) -- a quarter of the step on a
// 12 000-atom box, half a percent at 10^6 atoms.  Plain pointers on purpose: the passes read what earlier passes of the
// same kernel wrote, which the read-only data path would not see.
constexpr int SORT_THREADS = 512;
constexpr int SORT_SMALL_MAX_ATOMS = 32768, SORT_SMALL_CTAS = 32;   // small boxes: few CTAs, cheap barriers
__global__ void __launch_bounds__(SORT_THREADS) k_sort(SortArgs a, Universe u, unsigned short *cum) {
    if (a.go && *a.go != a.want) return;   // (every CTA takes the same way: nobody is left waiting at a barrier)
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    __shared__ int part[SORT_THREADS];
    const int t = blockIdx.x * SORT_THREADS + threadIdx.x, nt = gridDim.x * SORT_THREADS, n = a.n, ncell = a.grid.ncell;
    for (int c = t; c <= ncell; c += nt) { a.cell_count[c] = 0; a.cell_fill[c] = 0; }
    grid.sync();
    for (int i = t; i < n; i += nt) cell_key_one(i, a.xs, a.grid, a.key, a.cell_count, a.ctr);
    grid.sync();
    if (ncell <= 4 * SCAN_SLICE) {
        if (blockIdx.x == 0) scan_block(ncell, a.cell_count, a.cell_start, part);
    } else {   // large grids: sums of 4096-cell slices, their scan by one CTA, then every slice from its offset
        const int nslice = (ncell + SCAN_SLICE - 1) / SCAN_SLICE, tid = threadIdx.x;
        constexpr int PER = SCAN_SLICE / SORT_THREADS;   // cells per thread and slice
        for (int sl = blockIdx.x; sl < nslice; sl += gridDim.x) {
            int sum = 0;
            for (int k = 0; k < PER; ++k) { const int cc = sl * SCAN_SLICE + k * SORT_THREADS + tid; sum += cc < ncell ? a.cell_count[cc] : 0; }
            __syncthreads();
            part[tid] = sum;
            __syncthreads();
            for (int off = SORT_THREADS / 2; off > 0; off >>= 1) { if (tid < off) part[tid] += part[tid + off]; __syncthreads(); }
            if (tid == 0) a.scan_sums[sl] = part[0];
        }
        grid.sync();
        if (blockIdx.x == 0) scan_block(nslice, a.scan_sums, a.scan_offs, part);
        grid.sync();
        for (int sl = blockIdx.x; sl < nslice; sl += gridDim.x) {
            const int lo = sl * SCAN_SLICE + PER * tid;
            int cnt[PER], sum = 0;
#pragma unroll
            for (int k = 0; k < PER; ++k) { cnt[k] = lo + k < ncell ? a.cell_count[lo + k] : 0; sum += cnt[k]; }
            __syncthreads();
            part[tid] = sum;
            __syncthreads();
            for (int off = 1; off < SORT_THREADS; off <<= 1) {
                const int v = tid >= off ? part[tid - off] : 0;
                __syncthreads();
                part[tid] += v;
                __syncthreads();
            }
            int run = a.scan_offs[sl] + part[tid] - sum;
#pragma unroll
            for (int k = 0; k < PER; ++k) { if (lo + k < ncell) a.cell_start[lo + k] = run; run += cnt[k]; }
            if (lo <= ncell - 1 && ncell - 1 < lo + PER) a.cell_start[ncell] = run;
        }
    }
    grid.sync();
    for (int i = t; i < n; i += nt) scatter_one(i, a.key, a.orig, a.cell_start, a.cell_fill, a.tmp_orig, a.tmp_src);
    grid.sync();
    for (int c = t; c < ncell; c += nt) cell_sort_one(c, a.cell_start, a.tmp_orig, a.tmp_src);
    grid.sync();
    if (t == 0) { a.ctr->rebuilds += 1; a.ctr->last_build = a.want; }
    const int gnx = a.grid.gn[0], gny = a.grid.gn[1];
    for (int i = t; i < n; i += nt) {
        const int s = a.tmp_src[i], kk = a.key[s];
        a.cell_of[i] = pack_cell(kk % gnx, (kk / gnx) % gny, kk / (gnx * gny));
        const float4 x = a.xs[s];
        a.xs_t[i] = x; a.x_build[i] = x;
        a.vs_t[i] = a.vs[s]; a.xl_t[i] = a.xl[s]; a.lj_t[i] = a.lj[s]; a.hw_t[i] = a.hw[s]; a.mi_t[i] = a.mi[s];
        const int o = a.tmp_orig[i];
        a.orig_t[i] = o;
        a.sorted_of[o] = i;
    }
    grid.sync();
    for (int i = t; i < n; i += nt) {
        a.xs[i] = a.xs_t[i]; a.vs[i] = a.vs_t[i]; a.xl[i] = a.xl_t[i]; a.lj[i] = a.lj_t[i]; a.mi[i] = a.mi_t[i]; a.hw[i] = a.hw_t[i];
        a.orig[i] = a.orig_t[i];
    }
    if (!cum) return;
    // running sums of the cell universe (R-10c, ring C), one warp per home cell: reads cell_start only
    for (int h = t >> 5; h < ncell; h += nt >> 5) universe_cell(a.grid, u, a.cell_start, cum, a.ctr, h, t & 31);
}

// CTAs of a grid that fills the current device once with per_sm CTAs on every SM
static int resident_ctas(int per_sm) {
    static int sms[64] = {0};
    int dev = 0;
    cudaGetDevice(&dev);
    dev = std::max(0, std::min(dev, 63));
    if (!sms[dev]) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
        sms[dev] = v;
    }
    return sms[dev] * per_sm;
}

// uni_cum != NULL: the running sums of the cell universe are made too
void launch_sort(const SortArgs &a, const Universe &u, unsigned short *uni_cum, cudaStream_t st, int64_t *launches) {
    SortArgs aa = a;
    Universe uu = u;
    void *args[] = {(void *)&aa, (void *)&uu, (void *)&uni_cum};
    const int ctas = a.n <= SORT_SMALL_MAX_ATOMS ? SORT_SMALL_CTAS : resident_ctas(3);
    cudaLaunchCooperativeKernel((const void *)k_sort, dim3(ctas), dim3(SORT_THREADS), args, 0, st);
    *launches += 1;
}
int launch_universe_list(const SortGrid &g, const Universe &u, const int *cell_start, int home, int *out, int n,
                         cudaStream_t st, int64_t *launches) {
    if (n > 0) k_universe_list<<<(n + 127) / 128, 128, 0, st>>>(g, u, cell_start, home, n, out);
    *launches += 1;
    return 0;
}

void launch_build_rows(const Model &m, const SortGrid &g, const Row rows[N_ROWS], float rmax_all, const int *cell_start,
                       const float4 *xs, const float4 *xl, const float2 *lj, const float2 *hw, const int *orig, const int *sorted_of,
                       const int *excl_ptr, const int *excl_idx, Counters *ctr, int *cell_of, float far2, const int *go, int want,
                       cudaStream_t st, int64_t *launches) {
    RowSet rs;
    for (int k = 0; k < N_ROWS; ++k) rs.r[k] = rows[k];
    // stencil of cells within reach of a cell: gap between cells at offset o is (|o| - 1)_+ cell edges
    Stencil stn;
    double cs[3];
    for (int k = 0; k < 3; ++k) {
        cs[k] = (double)m.box[k] / g.gn[k];
        stn.R[k] = std::min(8, (int)std::ceil((double)rmax_all / cs[k]));  // init refuses grids that need more
    }
    const double r2 = (double)rmax_all * rmax_all;
    for (int a = 0; a < 17; ++a)
        for (int b = 0; b < 17; ++b) {
            double gz = std::max(a - 1, 0) * cs[2], gy = std::max(b - 1, 0) * cs[1];
            double rem = r2 - gz * gz - gy * gy;
            int v = -1;
            if (a <= stn.R[2] && b <= stn.R[1] && rem > 0.0) v = std::min(stn.R[0], (int)std::floor(std::sqrt(rem) / cs[0]) + 1);
            stn.xr[a * 17 + b] = (signed char)v;
        }
    int mask = 0;
    for (int k = 0; k < N_ROWS; ++k) mask |= rows[k].enabled ? (1 << k) : 0;
    // home cells per CTA: staging is shared by more atoms and the warps are better balanced, as long as the grid
    // still gives every SM several waves of CTAs
    // (measured on the 10^6-atom box: a home about 10 A long is best -- 5.6 ms per build against 6.0 at 7 A and 6.5 at 27 A)
    const int CX = std::max(1, std::min(std::min(BUILD_CX_MAX, (int)(11.0 / cs[0])), g.ncell / 4000));
    // FAST: staged coordinates relative to the cell centre, no minimum image in the inner loop (see k_build_rows)
    bool fast = true;
    for (int k = 0; k < 3; ++k) fast = fast && ((double)rmax_all + 0.5 * cs[k] * (k == 0 ? CX : 1) <= 0.5 * (double)m.box[k]) && m.box[k] <= 512.f;
    const int nblocks = ((g.gn[0] + CX - 1) / CX) * g.gn[1] * g.gn[2];
    const unsigned ngrid = (unsigned)std::min(nblocks, resident_ctas(7));
#define JB_BUILD(MASK)                                                                                                        \
    do {                                                                                                                      \
        if (fast) k_build_rows<MASK, true><<<ngrid, BUILD_THREADS, 0, st>>>(m, g, rs, stn, rmax_all, CX, cell_start, xs, xl, lj, hw, \
                                                                                     orig, sorted_of, excl_ptr, excl_idx, ctr, cell_of, far2, go, want, nblocks); \
        else k_build_rows<MASK, false><<<ngrid, BUILD_THREADS, 0, st>>>(m, g, rs, stn, rmax_all, CX, cell_start, xs, xl, lj, hw, \
                                                                                  orig, sorted_of, excl_ptr, excl_idx, ctr, cell_of, far2, go, want, nblocks);   \
    } while (0)
    switch (mask) {
        case 0x07: JB_BUILD(0x07); break;   // S A B     (JUMP with Coulomb and LJ jumps)
        case 0x27: JB_BUILD(0x27); break;   // S A B W   (Coulomb jumps only, R-13)
        case 0x10: JB_BUILD(0x10); break;   // F         (BAOAB comparator)
        case 0x01: JB_BUILD(0x01); break;   // S
        default: JB_BUILD(-1); break;
    }
#undef JB_BUILD
    *launches += 1;
}

}  // namespace jb
