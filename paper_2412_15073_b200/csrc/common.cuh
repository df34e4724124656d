// common.cuh -- shared declarations of the CUDA JUMP hot path (sm_100a).
// P:Lnnn = PAPER.md line, R-n = DESIGN.md reading.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/jump_b200.h"

namespace jb {

// R-1 constants (restated independently of the oracle)
constexpr double kKB = 1.987204259e-3;   // kcal/mol/K
constexpr double kCoulomb = 332.063713;  // kcal A / (mol e^2)
constexpr double kKcal = 418.4;          // (g/mol) A^2 ps^-2 per kcal/mol
constexpr float kInvSqrt2Pi = 0.3989422804014327f;
constexpr float kSqrt2Pi = 2.5066282746310002f;
constexpr float kTwoOverSqrtPi = 1.1283791670955126f;

// weight of a pair term: none, chi u (short), (1-chi) u (long), u (unsplit)
enum { W_NONE = 0, W_SHORT = 1, W_LONG = 2, W_FULL = 3 };
// row kinds (R-10c): S short list; A, B candidates of the jump rings [r_c-h, r_A), [r_A, r_M); F full list (BAOAB
// comparator); W LJ tail kept in F0 (R-13).  Ring C = [r_M, r_long) has no row: it draws from the cell universe.
enum { ROW_S = 0, ROW_A = 1, ROW_B = 2, ROW_UNUSED = 3, ROW_F = 4, ROW_W = 5, N_ROWS = 6 };
// device error bits
enum { ERR_OVERFLOW = 1, ERR_BOUND = 2, ERR_SKIN = 4, ERR_NAN = 8, ERR_EVENTS = 16 };

struct Row {
    int *idx;       // [n][cap] sorted indices, canonical order (R-10)
    int *cnt;       // [n]
    int cap;        // multiple of 32
    int lj_only;    // keep eps_i eps_j > 0 only
    // window of the pair (i, j) at a build (R-10c, mass-weighted skin): max(ra - s_ij, 0) <= d < rb + s_ij with
    // s_ij = (skin/2)(w_i + w_j); ra = 0: no lower edge
    float ra, rb;
    double ra_d, rb_d;   // the same in fp64 (edge decisions, R-17)
    int lo_plus;         // the lower edge is ra + s_ij instead (row W: the complement of row S)
    float r2max;         // (rb + skin w_max)^2: the farthest an entry can be at a build
    int enabled;
};

// device counters (one struct in global memory)
struct Counters {
    unsigned long long proposals, accepts, gt_attempts, expiries, n_events;
    unsigned int max_p_bits, max_gl_bits, max_disp2_bits;  // non-negative floats compared as uints
    unsigned int err;
    int max_row[N_ROWS];
    int go_step;            // step stamp of the last displacement trigger (k_update): the list kernels enqueued for that step run
    unsigned int rebuilds;  // sorts done (counted on the device: the host does not know which conditional ones ran)
    int last_build;         // step count at the last sort + list build (the list schedule counts from it, R-10c)
    int work_next[2], work_done[2];   // work queues of the resident-grid kernels (0 row build, 1 universe): next item, CTAs finished; 0 at rest
};

// Resident grid with a work queue: the CTAs of a grid that just fills the GPU take item numbers from a counter until
// they run out -- the load balance of one CTA per item without its launch cost, which for the list kernels is paid
// at EVERY step (they are always enqueued and return at once unless the step's displacement trigger armed them; a
// 131 072-CTA grid takes 70 us just to return).  The last CTA out puts the counters back to 0.
__device__ inline int work_fetch(Counters *ctr, int which, int *s_item) {
    __syncthreads();   // everybody has read the previous item (and is done with the shared memory of its work)
    if (threadIdx.x == 0) *s_item = atomicAdd(&ctr->work_next[which], 1);
    __syncthreads();
    return *s_item;
}
__device__ inline void work_leave(Counters *ctr, int which) {
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&ctr->work_done[which], 1) == (int)gridDim.x - 1) {
            ctr->work_next[which] = 0;
            ctr->work_done[which] = 0;
        }
    }
}

// constants of the physical model, passed by value to kernels
struct Model {
    int n;
    float box[3], inv_box[3];
    float rc, h, inv_h, rlo;      // r_c, h, 1/h, r_c - h
    float rc2, rlo2, rE2;         // squares
    double rlo2d;                 // (r_c - h)^2 in fp64 (switching argument, see chi_zone)
    float alpha, alpha2;          // Ewald alpha
    float beta;                   // 1/kT, (kcal/mol)^-1
    float eps_jump;               // epsilon; +inf -> BPS
    int eps_adaptive;             // eps(x) = eps_jump |F_ij(x)| (R-19)
    int combined;                 // step C' treats the whole long pair gradient, Coulomb + LJ, as one mechanism (R-22)
    float q_split;                // (min |q| + max |q|) / 2: atoms above it run the long chains (k_update's lane order)
    float qmaxG[3];               // qmax * G_Y, rings A, B, C   (L_Y,i = |q_i| * this, R-7)
    float GV4se[3];               // 4 sqrt(eps_max) GV_Y        (L^vdW_Y,i = sqrt(eps_i) * this)
    float ring2[4];               // squared ring edges (r_c-h)^2, r_A^2, r_M^2, r_long^2: ring Y = [ring2[Y], ring2[Y+1])
    double ring2d[4];             // the same in fp64 (an edge decision within RING_TIE is retaken in fp64, R-17)
    float half_skin2;             // (skin/2)^2
    float hs;                     // skin/2
    float Wc;                     // w_i = Wc / sqrt(beta m_i): mass weight of atom i's skin, m_i^-1/2 / mean(m^-1/2) (R-10c)
    float w_max;
    unsigned int key0, key1;      // Philox key = seed
};

// Philox4x32-10 (Salmon et al. SC'11), R-15: counter (atom, step, stream, block), key = seed.
__host__ __device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        // one 32 x 32 -> 64 product per multiplier (IMAD.WIDE on the device) gives both halves
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t h0 = (uint32_t)(p0 >> 32), l0 = (uint32_t)p0, h1 = (uint32_t)(p1 >> 32), l1 = (uint32_t)p1;
        uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// uniform in (0,1) with 24 significant bits, exact in fp32 and fp64 (R-15)
// = ((w >> 9) + 0.5) 2^-23, built in the mantissa: (1 + k 2^-23) - (1 - 2^-24) is exact (an odd multiple of 2^-24)
__device__ inline float u01(uint32_t w) { return __uint_as_float((w >> 9) | 0x3f800000u) - 0.99999994f; }

__device__ inline float wrap1(float x, float L, float invL) {
    x -= L * floorf(x * invL);
    if (x >= L) x -= L;
    if (x < 0.f) x = 0.f;
    return x;
}
// Minimum image of xi - xj, both in [0, L).  The periodic shift t L (t = -1, 0, 1) is applied so that it
// is EXACT: for t = +1 to xi (xi - L with xi in (L/2, L), Sterbenz), for t = -1 to xj (xj - L with xj in
// (L/2, L)); xi + L would round at ulp(2 L), an absolute error of ~4e-6 A at L = 62 A.  a - b then carries one
// rounding of the final difference only, and (double)a - (double)b is the exact image difference.
__device__ inline void image_pair1(float xi, float xj, float L, float invL, float &a, float &b) {
    float t = (xi - xj) * invL + 12582912.f;  // round to nearest integer by the 1.5 * 2^23 trick
    t -= 12582912.f;
    a = fmaf(-L, fmaxf(t, 0.f), xi);
    b = fmaf(L, fminf(t, 0.f), xj);
}
__device__ inline float min_image1(float xi, float xj, float L, float invL) {
    float a, b;
    image_pair1(xi, xj, L, invL, a, b);
    return a - b;
}

// Periodic image counters of an atom (NEXT-4: unwrapped trajectories for mean-square displacements): three
// 10-bit fields biased by 512, carried in the spare .w of the position residual xl and moved with it by the sort.
constexpr int kImgBias = 512;
__host__ __device__ inline int img_pack(int ix, int iy, int iz) {
    return ((ix + kImgBias) & 1023) | (((iy + kImgBias) & 1023) << 10) | (((iz + kImgBias) & 1023) << 20);
}
__host__ __device__ inline void img_unpack(int w, int &ix, int &iy, int &iz) {
    ix = (w & 1023) - kImgBias; iy = ((w >> 10) & 1023) - kImgBias; iz = ((w >> 20) & 1023) - kImgBias;
}

// erfc(x) exp(x^2) for 0 <= x <= 4.3 (alpha r never exceeds 3.8 (1 + skin / r_long)): degree-8 polynomial in
// t = 1 / (1 + x/2), a relative-weighted Chebyshev least-squares fit made for this file (max relative error
// 6e-8 in exact arithmetic, 2.6e-7 evaluated in fp32 -- the accuracy of erfcf).  erfc(alpha r) is then
// erfcx_poly(alpha r) * exp(-alpha^2 r^2) with the exponential the Coulomb derivative needs anyway:
// a third of the pair kernel's instructions were erfcf's.
// Bare MUFU approximations (no denormal or range fix-up code around them): rsqrt.approx / rcp.approx are good to
// 1-2 ulp and ex2.approx to 2 ulp on normal arguments, which is all the pair kernel feeds them (r^2 between 0.25 A^2 and
// the squared cutoff, exponents above -30); rsqrtf / exp2f wrap the same instructions in 4-6 more.
__device__ inline float rsqrt_fast(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ inline float rcp_fast(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ inline float ex2_fast(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

template <bool FAST = false>
__device__ inline float erfcx_poly(float x) {
    // rcp.approx: 1 ulp, the IEEE reciprocal costs 8 instructions
    float t = FAST ? rcp_fast(fmaf(0.5f, x, 1.f)) : __fdividef(1.f, fmaf(0.5f, x, 1.f));
    float p = -4.621402847e-02f;
    p = fmaf(p, t, 3.202601290e-01f);
    p = fmaf(p, t, -8.488328818e-01f);
    p = fmaf(p, t, 9.638187580e-01f);
    p = fmaf(p, t, -3.656822066e-01f);
    p = fmaf(p, t, 4.560536203e-01f);
    p = fmaf(p, t, 2.321311377e-01f);
    p = fmaf(p, t, 2.888640654e-01f);
    p = fmaf(p, t, -3.985373802e-04f);
    return p;
}

// chi (R-3): quintic smootherstep on [rc-h, rc]; returns chi, writes dchi/dr.
// Outside the switching zone chi is 0 or 1 and nothing else is computed.  Inside it the argument
// u = (r - r_lo)/h is formed as (r^2 - r_lo^2) / (h (r + r_lo)) with r^2 - r_lo^2 in fp64 from the exact
// coordinate differences (a - b of image_pair1): a plain fp32 r - r_lo carries an absolute error
// of ~3e-7 A that chi'' u_C (~10 kcal/mol/A^2) turns into ~3e-6 per pair -- the largest error of the long
// force and of the acceptance probabilities p (R-16, R-17).
// EXACT = false (the pair kernel, whose output is a sum over ~100 pairs compared with the whole gradient): the same
// ratio with r^2 - r_lo^2 in fp32, 6e-7 in u -- the fp64 conversions and FMAs were 15 % of that kernel's instructions.
template <bool EXACT>
__device__ inline float chi_zone(float ax, float ay, float az, float bx, float by, float bz, float r2, float r,
                                 const Model &m, float &dchi) {
    if (EXACT) {
        if (r2 <= m.rlo2) { dchi = 0.f; return 1.f; }
        if (r2 >= m.rc2) { dchi = 0.f; return 0.f; }
    }   // (the fp32 form needs no branch: the clamp of u to [0, 1] gives chi = 1, 0 and chi' = 0 outside the zone)
    float num;
    if (EXACT) {
        double dx = (double)ax - (double)bx, dy = (double)ay - (double)by, dz = (double)az - (double)bz;
        num = (float)fma(dx, dx, fma(dy, dy, fma(dz, dz, -m.rlo2d)));
    } else num = r2 - m.rlo2;
    float u = __fdividef(num * m.inv_h, r + m.rlo);
    u = fminf(fmaxf(u, 0.f), 1.f);
    float omu = 1.f - u;
    dchi = -30.f * u * u * omu * omu * m.inv_h;
    return 1.f - u * u * u * (10.f - 15.f * u + 6.f * u * u);
}

// ---------------------------------------------------------------------------------------------
// host-visible launchers (one per .cu file group)
// ---------------------------------------------------------------------------------------------
struct SortGrid {
    int gn[3];
    double scale[3];  // gn / box (fp64: the cell of an atom is decided in the oracle's precision, R-10)
    int ncell;
    int reach[3];     // cells to visit on each side for the largest enabled row
};

// Cell universe of jump ring C (R-10c): the atoms of every contract-grid cell within reach r_long + skin of the home
// cell, in ascending (cell key, original index) order = a list of contiguous runs of the cell-sorted atom array, one or
// two per (z, y) cell row of the stencil.  Per home cell the library keeps the running sums of the row lengths
// (cum[h][p], p = mz * cnt_y + my in ascending (z, y); cum[h][nrow] = size of the universe).
struct Universe {
    int R[3];                 // stencil reach in cells per dimension
    int cnt[3];               // cells covered per dimension: min(2 R + 1, gn)
    int nrow;                 // cnt[2] * cnt[1]
    int stride;               // entries per home cell in cum (nrow + 1, padded)
    int inv_cnt1;             // ceil(65536 / cnt[1]): row index -> (mz, my) without a division
    signed char xr[17 * 17];  // [|oz| * 17 + |oy|] -> largest |ox| within reach, -1: (z, y) cell row out of reach
    const unsigned short *cum;
    const int *cell_of;       // home cell of each sorted atom, packed (pack_cell)
};

// m-th value, in ascending order, of the cyclic cell range [start, start+cnt) mod gn
__host__ __device__ inline int cyc_val(int m, int start, int cnt, int gn) {
    int w = start + cnt - gn;
    if (w < 0) w = 0;
    return m < w ? m : start + m - w;
}
__host__ __device__ inline int cyc_off(int val, int c, int gn) {
    int o = val - c;
    if (2 * o > gn) o -= gn;
    else if (2 * o < -gn) o += gn;
    return o;
}
// home cell of an atom, packed: cx | cy << 10 | cz << 20 (at most 1023 cells per edge)
__host__ __device__ inline int pack_cell(int cx, int cy, int cz) { return cx | (cy << 10) | (cz << 20); }
// The runs of stencil row (mz, my) of home cell (cx, cy, cz): sorted atoms [b0, b0 + n0) (cells wrapped to the low end
// of the x axis, first in key order) then [b1, b1 + n1).  Shared by the table build (sort_build.cu) and the draw
// (chains.cuh).  No integer division: every wrap is a conditional add.
__device__ inline void universe_row(const SortGrid &g, const Universe &u, const int *__restrict__ cell_start, int cx, int cy,
                                    int cz, int mz, int my, int &b0, int &n0, int &b1, int &n1) {
    b0 = n0 = b1 = n1 = 0;
    int sz = 0, sy = 0;
    if (u.cnt[2] != g.gn[2]) { sz = cz - u.R[2]; if (sz < 0) sz += g.gn[2]; }
    if (u.cnt[1] != g.gn[1]) { sy = cy - u.R[1]; if (sy < 0) sy += g.gn[1]; }
    const int zc = cyc_val(mz, sz, u.cnt[2], g.gn[2]), yc = cyc_val(my, sy, u.cnt[1], g.gn[1]);
    int oz = cyc_off(zc, cz, g.gn[2]), oy = cyc_off(yc, cy, g.gn[1]);
    oz = oz < 0 ? -oz : oz; oy = oy < 0 ? -oy : oy;
    const int xm = u.xr[oz * 17 + oy];
    if (xm < 0) return;
    const int rowbase = (zc * g.gn[1] + yc) * g.gn[0];
    if (2 * xm + 1 >= g.gn[0]) {
        b1 = cell_start[rowbase]; n1 = cell_start[rowbase + g.gn[0]] - b1;
    } else {
        int xs0 = cx - xm;
        if (xs0 < 0) xs0 += g.gn[0];
        const int xc = 2 * xm + 1;
        int w = xs0 + xc - g.gn[0];
        if (w < 0) w = 0;
        if (w > 0) { b0 = cell_start[rowbase]; n0 = cell_start[rowbase + w] - b0; }
        b1 = cell_start[rowbase + xs0]; n1 = cell_start[rowbase + xs0 + xc - w] - b1;
    }
}

// k-th atom (sorted index) of the universe of the home cell `hp` (packed coordinates): a fixed-length bisection on the
// running sums of the stencil rows (nine dependent 2-byte loads from a few cache lines), then the row's one or two runs
__device__ inline int universe_pick(const SortGrid &g, const Universe &u, const int *__restrict__ cell_start, int hp, int k) {
    const int cx = hp & 1023, cy = (hp >> 10) & 1023, cz = hp >> 20;
    const int h = (cz * g.gn[1] + cy) * g.gn[0] + cx;
    const unsigned short *__restrict__ cum = u.cum + (size_t)h * u.stride;
    int lo = 0;   // last row with cum[row] <= k
#pragma unroll
    for (int step = 256; step > 0; step >>= 1) {
        const int t = lo + step;
        if (t < u.nrow && (int)cum[t] <= k) lo = t;
    }
    const int mz = (lo * u.inv_cnt1) >> 16, my = lo - mz * u.cnt[1];   // lo / cnt[1] by a reciprocal (lo < 512, cnt[1] <= 17)
    int b0, n0, b1, n1;
    universe_row(g, u, cell_start, cx, cy, cz, mz, my, b0, n0, b1, n1);
    const int kk = k - (int)cum[lo];
    return kk < n0 ? b0 + kk : b1 + (kk - n0);
}
__device__ inline int universe_size(const SortGrid &g, const Universe &u, int hp) {
    const int h = ((hp >> 20) * g.gn[1] + ((hp >> 10) & 1023)) * g.gn[0] + (hp & 1023);
    return (int)u.cum[(size_t)h * u.stride + u.nrow];
}

struct Topo {  // per-atom CSR of bonded terms in ORIGINAL indices (device)
    const int *bptr, *bother;   // bonds: partner atom
    const float *bk, *br0;
    const int *aptr, *arole, *aa, *ab;  // angles: my role (0 end i, 1 vertex, 2 end k) and the two other atoms
    const float *ak, *at0;
};

constexpr float RING_TIE = 4e-3f;   // A^2: an fp32 r^2 this close to a ring edge is re-decided in fp64 (R-17)

// Bonded terms of one kind of small molecule (<= 3 atoms), local atom numbers 0..2 (forces.cu: k_bonded_mol)
struct MolType {
    int nb, na;
    int bp[3], bq[3];
    float bk[3], br0[3];
    int ai[3], av[3], ak_[3];   // angle: end, vertex, end
    float ak[3], at0[3];
};
struct Bonded {
    int nmol;                 // small molecules: one thread each
    const int4 *mols;         // (a0, a1, a2 original indices or -1, type)
    const MolType *types;
    int nbig;                 // atoms of larger components: per-atom CSR (Topo)
    const int *big_atoms;     // original indices
};

struct Phase {      // one half-phase of velocity updates at frozen x
    int kind;       // 0 none, 1 kick (B), 2 jump chains
    float H;        // duration, ps
    int use_grad;   // acceleration a = -M^-1 (ga + gb) else 0
    int reverse;    // J' before C'
    int bkick;      // kind 2 only: 0 = the chains run under the acceleration (step C'); 1 / 2 = B J / J B:
                    // the kick H a apart, before / after chains on a piecewise constant velocity
    int coul, lj;   // which chains run (kind 2)
    int streamC, streamJ;
    unsigned int step;
};

}  // namespace jb
