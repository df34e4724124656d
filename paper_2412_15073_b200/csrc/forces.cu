// forces.cu -- bonded gradient and switched pair gradient (a5, a10).
//
// Pair term (R-2, R-3, R-8):
//   u_C(r) = C q_i q_j erfc(alpha r)/r,  u_LJ(r) = 4 eps_ij [(s_ij/r)^12 - (s_ij/r)^6],
//   short part chi(r) u, long part (1-chi(r)) u, unsplit u; 0 beyond r_long.
// Every output is a GRADIENT piece (R-4).  One warp per atom over a full (both directions) row:
// the 32 lanes take 32 consecutive row entries (one coalesced 128-byte index load), gather x_j,
// accumulate in registers and reduce by shuffles -- no floating-point atomics, deterministic.
#include "launch.h"

namespace jb {

template <int W>
__device__ inline float weighted_du(float chi, float dchi, float u, float du) {
    if (W == W_FULL) return du;
    if (W == W_SHORT) return chi * du + dchi * u;  // d/dr [chi u]
    return (1.f - chi) * du - dchi * u;             // d/dr [(1-chi) u]
}
template <int W>
__device__ inline float weighted_u(float chi, float u) {
    if (W == W_FULL) return u;
    return W == W_SHORT ? chi * u : (1.f - chi) * u;
}

// CTAs of two warps: rows differ in length, and small CTAs leave an SM's slots sooner (256 threads: 630 us at 10^6
// atoms, 128: 617, 64: 612)
constexpr int PAIR_THREADS = 64;

// One warp per atom over its row (entries: sorted index of j, bit 31 set when j carries LJ).
// INTERIOR: the atom is farther than the row's reach + 2 skins from every box face, so no partner of its row can
// be a periodic image: plain differences, no minimum image in the inner loop.
template <int WC, int WLJ, bool ENERGY, bool INTERIOR>
__device__ inline void pair_warp(const Model &m, const Row &row, const float4 *__restrict__ xs,
                                 const float2 *__restrict__ lj, float4 *__restrict__ out, int accumulate, int i, int lane,
                                 const float4 xi) {
    const unsigned full = 0xffffffffu;
    const float qi = (float)kCoulomb * xi.w;
    const float2 lji = lj[i];
    const float cutC2 = (WC == W_SHORT) ? m.rc2 : m.rE2, cutL2 = (WLJ == W_SHORT) ? m.rc2 : m.rE2;
    const float cut2 = (WC == W_NONE) ? cutL2 : ((WLJ == W_NONE) ? cutC2 : fmaxf(cutC2, cutL2));
    const bool do_lj = (WLJ != W_NONE) && lji.y > 0.f;
    // both terms end at the same cutoff: the per-term tests after the common one are dropped at compile time
    constexpr bool SAME_CUT = WC == W_NONE || WLJ == W_NONE || ((WC == W_SHORT) == (WLJ == W_SHORT));
    constexpr bool NEED_CHI = WC == W_SHORT || WC == W_LONG || WLJ == W_SHORT || WLJ == W_LONG;
    const float na2l = -m.alpha2 * 1.4426950408889634f;   // exp(-alpha^2 r^2) = 2^(na2l r^2)
    const float kq = kTwoOverSqrtPi * m.alpha;
    const float u_b = -m.rlo * m.inv_h;                   // switching argument u = r / h - r_lo / h
    const int cnt = row.cnt[i];
    const int *__restrict__ ridx = row.idx + (size_t)i * row.cap;
    float fx = 0.f, fy = 0.f, fz = 0.f, en = 0.f;
    // software pipeline: the index two iterations ahead and the position one iteration ahead are in flight while
    // the current entry is evaluated (the gathers' L1/L2 latency was the kernel's largest stall)
    int j1 = lane < cnt ? ridx[lane] : 0, j2 = lane + 32 < cnt ? ridx[lane + 32] : 0;
    float4 x1 = xs[j1 & 0x7fffffff];
    for (int k = lane; k < cnt; k += 32) {
        const int jraw = j1;
        const float4 xj = x1;
        j1 = j2;
        x1 = xs[j1 & 0x7fffffff];
        j2 = k + 64 < cnt ? ridx[k + 64] : 0;
        float dx, dy, dz;
        if (INTERIOR) { dx = xi.x - xj.x; dy = xi.y - xj.y; dz = xi.z - xj.z; }
        else {
            dx = min_image1(xi.x, xj.x, m.box[0], m.inv_box[0]);
            dy = min_image1(xi.y, xj.y, m.box[1], m.inv_box[1]);
            dz = min_image1(xi.z, xj.z, m.box[2], m.inv_box[2]);
        }
        const float r2 = dx * dx + dy * dy + dz * dz;
        if (r2 >= cut2) continue;
        const float rinv = rsqrt_fast(r2), r = r2 * rinv;
        float fr = 0.f, chi = 1.f, dchi = 0.f;
        if (NEED_CHI) {   // chi (R-3): quintic smootherstep on [r_c - h, r_c]; the clamp gives 1, 0 and chi' = 0 outside
            const float u = __saturatef(fmaf(r, m.inv_h, u_b)), omu = 1.f - u, u2 = u * u;
            dchi = -30.f * m.inv_h * (u2 * (omu * omu));
            chi = fmaf(-(u2 * u), fmaf(u, fmaf(6.f, u, -15.f), 10.f), 1.f);
        }
        if (WC != W_NONE && (SAME_CUT || r2 < cutC2)) {
            const float qq = qi * xj.w;
            const float ex = ex2_fast(na2l * r2), e = ex * erfcx_poly<true>(m.alpha * r);   // erfc(alpha r)
            const float u = qq * e * rinv;
            const float du = -(u + qq * kq * ex) * rinv;  // u'
            fr += weighted_du<WC>(chi, dchi, u, du);
            if (ENERGY) en += weighted_u<WC>(chi, u);
        }
        if (do_lj && jraw < 0 && (SAME_CUT || r2 < cutL2)) {
            const float2 ljj = lj[jraw & 0x7fffffff];
            const float s = lji.x * ljj.x * rinv, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
            const float e4 = lji.y * ljj.y;  // 4 eps_ij (R-8: geometric mixing)
            const float u = e4 * (s12 - s6);
            const float du = e4 * (6.f * s6 - 12.f * s12) * rinv;
            fr += weighted_du<WLJ>(chi, dchi, u, du);
            if (ENERGY) en += weighted_u<WLJ>(chi, u);
        }
        const float s = fr * rinv;
        fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        fx += __shfl_xor_sync(full, fx, off);
        fy += __shfl_xor_sync(full, fy, off);
        fz += __shfl_xor_sync(full, fz, off);
        if (ENERGY) en += __shfl_xor_sync(full, en, off);
    }
    if (lane == 0) {
        float4 o = make_float4(fx, fy, fz, 0.5f * en);
        if (accumulate) { float4 p = out[i]; o.x += p.x; o.y += p.y; o.z += p.z; o.w += p.w; }
        out[i] = o;
    }
}

template <int WC, int WLJ, bool ENERGY>
__global__ void __launch_bounds__(PAIR_THREADS) k_pair(Model m, Row row, float margin, const float4 *__restrict__ xs,
                                              const float2 *__restrict__ lj, float4 *__restrict__ out, int accumulate) {
    int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= m.n) return;
    const float4 xi = xs[i];
    // margin = reach of the row + 2 skins (a partner was within reach at the build; both atoms moved < skin since)
    const bool interior = xi.x > margin && xi.x < m.box[0] - margin && xi.y > margin && xi.y < m.box[1] - margin &&
                          xi.z > margin && xi.z < m.box[2] - margin;
    if (interior) pair_warp<WC, WLJ, ENERGY, true>(m, row, xs, lj, out, accumulate, i, lane, xi);
    else pair_warp<WC, WLJ, ENERGY, false>(m, row, xs, lj, out, accumulate, i, lane, xi);
}

// Harmonic bonds k (r-r0)^2 and angles k (theta-theta0)^2 (R-2), in fp64: at the equilibrium geometry r - r0 and
// theta - theta0 cancel to rounding, and the gradient there is compared with the fp64 oracle's relative to its own
// (tiny) size.  Every term is evaluated ONCE:
//   k_bonded_mol  one thread per small molecule (a connected component of the bonded graph with at most three atoms:
//                 water), its bonds and angles from a per-type table, the gradients of its atoms written directly --
//                 each atom belongs to one molecule, so there is nothing to reduce and nothing atomic;
//   k_bonded_csr  the atoms of larger components (chains), one thread per atom over the terms it takes part in.
__device__ inline double min_image_d(double xi, double xj, float L) {
    double d = xi - xj, Ld = (double)L;
    return d - Ld * rint(d / Ld);
}

struct D3 { double x, y, z; };
__device__ inline D3 full_pos(const float4 *__restrict__ xs, const float4 *__restrict__ xl, int i) {
    float4 a = xs[i], b = xl[i];  // x = hi + lo (the A steps integrate in fp64, see update.cu)
    return D3{(double)a.x + (double)b.x, (double)a.y + (double)b.y, (double)a.z + (double)b.z};
}
__device__ inline D3 image_diff(const Model &m, const D3 &a, const D3 &b) {
    return D3{min_image_d(a.x, b.x, m.box[0]), min_image_d(a.y, b.y, m.box[1]), min_image_d(a.z, b.z, m.box[2])};
}
// gradient of k (theta - theta0)^2 with respect to the two ends (u = end1 - vertex, w = end2 - vertex); the vertex takes
// minus their sum
__device__ inline double angle_term(const D3 &u, const D3 &w, double k, double t0, D3 &g1, D3 &g2) {
    const double lu = sqrt(u.x * u.x + u.y * u.y + u.z * u.z), lw = sqrt(w.x * w.x + w.y * w.y + w.z * w.z);
    double ct = (u.x * w.x + u.y * w.y + u.z * w.z) / (lu * lw);
    ct = fmin(1.0, fmax(-1.0, ct));
    const double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12);
    const double dth = th - t0, dU = 2.0 * k * dth;
    const double c1 = -dU / (lu * st), c2 = -dU / (lw * st);
    g1 = D3{c1 * (w.x / lw - ct * u.x / lu), c1 * (w.y / lw - ct * u.y / lu), c1 * (w.z / lw - ct * u.z / lu)};
    g2 = D3{c2 * (u.x / lu - ct * w.x / lw), c2 * (u.y / lu - ct * w.y / lw), c2 * (u.z / lu - ct * w.z / lw)};
    return k * dth * dth;
}

__device__ inline D3 sel3(const D3 x[3], int k) { return k == 0 ? x[0] : (k == 1 ? x[1] : x[2]); }

__global__ void __launch_bounds__(128) k_bonded_mol(Model m, int nmol, const int4 *__restrict__ mols, const MolType *__restrict__ types,
                                                    const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                    const int *__restrict__ sorted_of, float4 *__restrict__ out_bond) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nmol) return;
    const int4 a = mols[t];                      // original indices of the atoms (-1: none), type
    const MolType ty = types[a.w];
    int idx[3] = {sorted_of[a.x], a.y >= 0 ? sorted_of[a.y] : -1, a.z >= 0 ? sorted_of[a.z] : -1};
    D3 x[3], g[3];
    double e[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        x[k] = idx[k] >= 0 ? full_pos(xs, xl, idx[k]) : D3{0.0, 0.0, 0.0};
        g[k] = D3{0.0, 0.0, 0.0};
    }
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        if (b >= ty.nb) break;
        const int p = ty.bp[b], q = ty.bq[b];
        const D3 d = image_diff(m, sel3(x, p), sel3(x, q));
        const double r = sqrt(d.x * d.x + d.y * d.y + d.z * d.z), dr = r - (double)ty.br0[b], k = (double)ty.bk[b];
        const double f = 2.0 * k * dr / r;
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) {   // (static indexing keeps x, g in registers)
            const double sgn = k2 == p ? 1.0 : (k2 == q ? -1.0 : 0.0);
            g[k2].x += sgn * f * d.x; g[k2].y += sgn * f * d.y; g[k2].z += sgn * f * d.z;
            e[k2] += (sgn != 0.0 ? 0.5 : 0.0) * k * dr * dr;
        }
    }
#pragma unroll
    for (int an = 0; an < 3; ++an) {
        if (an >= ty.na) break;
        const int i1 = ty.ai[an], v = ty.av[an], i2 = ty.ak_[an];
        const D3 xe1 = sel3(x, i1), xv = sel3(x, v), xe2 = sel3(x, i2);
        D3 g1, g2;
        const double en = angle_term(image_diff(m, xe1, xv), image_diff(m, xe2, xv), (double)ty.ak[an], (double)ty.at0[an], g1, g2);
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) {
            const double s1 = k2 == i1 ? 1.0 : 0.0, s2 = k2 == i2 ? 1.0 : 0.0, sv = k2 == v ? -1.0 : 0.0;
            g[k2].x += s1 * g1.x + s2 * g2.x + sv * (g1.x + g2.x);
            g[k2].y += s1 * g1.y + s2 * g2.y + sv * (g1.y + g2.y);
            g[k2].z += s1 * g1.z + s2 * g2.z + sv * (g1.z + g2.z);
            e[k2] += (k2 == i1 || k2 == i2 || k2 == v) ? en * (1.0 / 3.0) : 0.0;
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
        if (idx[k] >= 0) out_bond[idx[k]] = make_float4((float)g[k].x, (float)g[k].y, (float)g[k].z, (float)e[k]);
}

// atoms of larger components: one thread per listed atom (original index) over its CSR of terms
__global__ void __launch_bounds__(128) k_bonded_csr(Model m, Topo t, int natoms, const int *__restrict__ atoms,
                                                    const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                    const int *__restrict__ sorted_of, float4 *__restrict__ out_bond) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= natoms) return;
    const int o = atoms[q], i = sorted_of[o];
    const D3 xi = full_pos(xs, xl, i);
    double gx = 0., gy = 0., gz = 0., en = 0.;
    for (int b = t.bptr[o]; b < t.bptr[o + 1]; ++b) {
        const D3 d = image_diff(m, xi, full_pos(xs, xl, sorted_of[t.bother[b]]));
        const double r = sqrt(d.x * d.x + d.y * d.y + d.z * d.z), dr = r - (double)t.br0[b], k = (double)t.bk[b];
        const double f = 2.0 * k * dr / r;
        gx += f * d.x; gy += f * d.y; gz += f * d.z;
        en += 0.5 * k * dr * dr;
    }
    for (int a = t.aptr[o]; a < t.aptr[o + 1]; ++a) {
        // role 1: I am the vertex, (aa, ab) are the ends; else I am an end, aa = vertex, ab = other end
        const int role = t.arole[a];
        const D3 xa = full_pos(xs, xl, sorted_of[t.aa[a]]), xb = full_pos(xs, xl, sorted_of[t.ab[a]]);
        const D3 xv = role == 1 ? xi : xa, xe1 = role == 1 ? xa : xi;
        D3 g1, g2;
        const double e3 = angle_term(image_diff(m, xe1, xv), image_diff(m, xb, xv), (double)t.ak[a], (double)t.at0[a], g1, g2);
        if (role == 1) { gx -= g1.x + g2.x; gy -= g1.y + g2.y; gz -= g1.z + g2.z; }
        else { gx += g1.x; gy += g1.y; gz += g1.z; }
        en += e3 * (1.0 / 3.0);
    }
    out_bond[i] = make_float4((float)gx, (float)gy, (float)gz, (float)en);
}

// out[orig[i]] = f[i].xyz  (sorted -> caller order)
__global__ void k_unsort3(int n, const float4 *__restrict__ f, const float4 *__restrict__ f2, const int *__restrict__ orig,
                          float *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = f[i];
    if (f2) { const float4 w = f2[i]; v.x += w.x; v.y += w.y; v.z += w.z; }
    int o = orig[i];
    out[3 * o] = v.x; out[3 * o + 1] = v.y; out[3 * o + 2] = v.z;
}

// number of ordered row entries currently within r_cut (measurement: algorithmic pairs per launch)
__global__ void k_count_pairs(Model m, Row row, const float4 *__restrict__ xs, float rc2, unsigned long long *out) {
    int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= m.n) return;
    const float4 xi = xs[i];
    const int cnt = row.cnt[i];
    const int *__restrict__ ridx = row.idx + (size_t)i * row.cap;
    unsigned c = 0;
    for (int k = lane; k < cnt; k += 32) {
        float4 xj = xs[ridx[k] & 0x7fffffff];
        float dx = min_image1(xi.x, xj.x, m.box[0], m.inv_box[0]);
        float dy = min_image1(xi.y, xj.y, m.box[1], m.inv_box[1]);
        float dz = min_image1(xi.z, xj.z, m.box[2], m.inv_box[2]);
        c += (dx * dx + dy * dy + dz * dz < rc2) ? 1u : 0u;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    if (lane == 0 && c) atomicAdd(out, (unsigned long long)c);
}
void launch_count_pairs(const Model &m, const Row &row, const float4 *xs, float rc2, unsigned long long *out,
                        cudaStream_t st, int64_t *launches) {
    const int B = 256;
    k_count_pairs<<<(unsigned)(((long long)m.n * 32 + B - 1) / B), B, 0, st>>>(m, row, xs, rc2, out);
    *launches += 1;
}

template <int WC, int WLJ>
static void pair_dispatch(const Model &m, const Row &row, const float4 *xs, const float2 *lj, float4 *out, int accumulate,
                          bool energy, cudaStream_t st) {
    const int B = PAIR_THREADS;
    unsigned grid = (unsigned)(((long long)m.n * 32 + B - 1) / B);
    const float margin = sqrtf(row.r2max) + 2.f * m.hs * m.w_max * 2.f;   // farthest entry at a build + what two atoms may move
    if (energy) k_pair<WC, WLJ, true><<<grid, B, 0, st>>>(m, row, margin, xs, lj, out, accumulate);
    else k_pair<WC, WLJ, false><<<grid, B, 0, st>>>(m, row, margin, xs, lj, out, accumulate);
}

int launch_pair(const Model &m, const Row &row, int wC, int wLJ, const float4 *xs, const float2 *lj, float4 *out,
                int accumulate, bool energy, cudaStream_t st, int64_t *launches) {
    *launches += 1;
#define JB_CASE(a, b) \
    if (wC == a && wLJ == b) { pair_dispatch<a, b>(m, row, xs, lj, out, accumulate, energy, st); return 0; }
    JB_CASE(W_SHORT, W_SHORT) JB_CASE(W_SHORT, W_FULL) JB_CASE(W_NONE, W_FULL) JB_CASE(W_FULL, W_FULL)
    JB_CASE(W_LONG, W_LONG) JB_CASE(W_LONG, W_NONE) JB_CASE(W_SHORT, W_NONE)
#undef JB_CASE
    *launches -= 1;
    return -1;
}

void launch_bonded(const Model &m, const Topo &t, const Bonded &b, const float4 *xs, const float4 *xl, const int *sorted_of,
                   float4 *out_bond, cudaStream_t st, int64_t *launches) {
    const int B = 128;
    if (b.nmol > 0) {
        k_bonded_mol<<<(b.nmol + B - 1) / B, B, 0, st>>>(m, b.nmol, b.mols, b.types, xs, xl, sorted_of, out_bond);
        *launches += 1;
    }
    if (b.nbig > 0) {
        k_bonded_csr<<<(b.nbig + B - 1) / B, B, 0, st>>>(m, t, b.nbig, b.big_atoms, xs, xl, sorted_of, out_bond);
        *launches += 1;
    }
}

void launch_unsort3(int n, const float4 *f, const float4 *f2, const int *orig, float *out, cudaStream_t st, int64_t *launches) {
    const int B = 256;
    k_unsort3<<<(n + B - 1) / B, B, 0, st>>>(n, f, f2, orig, out);
    *launches += 1;
}

}  // namespace jb
