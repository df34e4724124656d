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

template <int WC, int WLJ, bool ENERGY>
__device__ inline void pair_warp(const Model &m, const Row &row, const float4 *__restrict__ xs,
                                 const float2 *__restrict__ lj, float4 *__restrict__ out, int accumulate, int i, int lane) {
    const unsigned full = 0xffffffffu;
    const float4 xi = xs[i];
    const float qi = (float)kCoulomb * xi.w;
    const float2 lji = lj[i];
    const float cutC2 = (WC == W_SHORT) ? m.rc2 : m.rE2, cutL2 = (WLJ == W_SHORT) ? m.rc2 : m.rE2;
    const float cut2 = (WC == W_NONE) ? cutL2 : ((WLJ == W_NONE) ? cutC2 : fmaxf(cutC2, cutL2));
    const bool do_lj = (WLJ != W_NONE) && lji.y > 0.f;
    // both terms end at the same cutoff: the per-term tests after the common one are dropped at compile time
    constexpr bool SAME_CUT = WC == W_NONE || WLJ == W_NONE || ((WC == W_SHORT) == (WLJ == W_SHORT));
    const int cnt = row.cnt[i];
    const int *__restrict__ ridx = row.idx + (size_t)i * row.cap;
    float fx = 0.f, fy = 0.f, fz = 0.f, en = 0.f;
    // software pipeline: the index two iterations ahead and the position one iteration ahead are in flight while
    // the current entry is evaluated (the gathers' L1/L2 latency was the kernel's largest stall)
    int j1 = lane < cnt ? ridx[lane] : 0, j2 = lane + 32 < cnt ? ridx[lane + 32] : 0;
    float4 x1 = xs[j1];
    for (int k = lane; k < cnt; k += 32) {
        const int j = j1;
        const float4 xj = x1;
        j1 = j2;
        x1 = xs[j1];
        j2 = k + 64 < cnt ? ridx[k + 64] : 0;
        float ax, ay, az, bx, by, bz;
        image_pair1(xi.x, xj.x, m.box[0], m.inv_box[0], ax, bx);
        image_pair1(xi.y, xj.y, m.box[1], m.inv_box[1], ay, by);
        image_pair1(xi.z, xj.z, m.box[2], m.inv_box[2], az, bz);
        float dx = ax - bx, dy = ay - by, dz = az - bz;
        float r2 = dx * dx + dy * dy + dz * dz;
        if (r2 >= cut2) continue;
        float rinv = rsqrtf(r2), r = r2 * rinv;
        float fr = 0.f, chi = 1.f, dchi = 0.f;
        if (WC == W_SHORT || WC == W_LONG || WLJ == W_SHORT || WLJ == W_LONG) chi = chi_zone<false>(ax, ay, az, bx, by, bz, r2, r, m, dchi);
        if (WC != W_NONE && (SAME_CUT || r2 < cutC2)) {
            float qq = qi * xj.w;
            float ex = expf(-m.alpha2 * r2), e = ex * erfcx_poly(m.alpha * r);
            float u = qq * e * rinv;
            float du = -(u + qq * kTwoOverSqrtPi * m.alpha * ex) * rinv;  // u'
            fr += weighted_du<WC>(chi, dchi, u, du);
            if (ENERGY) en += weighted_u<WC>(chi, u);
        }
        if (do_lj && (SAME_CUT || r2 < cutL2)) {
            float2 ljj = lj[j];
            if (ljj.y > 0.f) {
                float s = lji.x * ljj.x * rinv, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
                float e4 = lji.y * ljj.y;  // 4 eps_ij (R-8: geometric mixing)
                float u = e4 * (s12 - s6);
                float du = e4 * (6.f * s6 - 12.f * s12) * rinv;
                fr += weighted_du<WLJ>(chi, dchi, u, du);
                if (ENERGY) en += weighted_u<WLJ>(chi, u);
            }
        }
        float s = fr * rinv;
        fx += s * dx; fy += s * dy; fz += s * dz;
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
__global__ void __launch_bounds__(256) k_pair(Model m, Row row, const float4 *__restrict__ xs,
                                              const float2 *__restrict__ lj, float4 *__restrict__ out, int accumulate) {
    int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i >= m.n) return;
    pair_warp<WC, WLJ, ENERGY>(m, row, xs, lj, out, accumulate, i, lane);
}

// Harmonic bonds k (r-r0)^2 and angles k (theta-theta0)^2 (R-2), one thread per atom over the terms
// the atom takes part in; evaluated in fp64 (a few hundred flops per atom) because r - r0 cancels.
__device__ inline double min_image_d(double xi, double xj, float L) {
    double d = xi - xj, Ld = (double)L;
    return d - Ld * rint(d / Ld);
}

struct D3 { double x, y, z; };
__device__ inline D3 full_pos(const float4 *__restrict__ xs, const float4 *__restrict__ xl, int i) {
    float4 a = xs[i], b = xl[i];  // x = hi + lo (the A steps integrate in fp64, see update.cu)
    return D3{(double)a.x + (double)b.x, (double)a.y + (double)b.y, (double)a.z + (double)b.z};
}

__global__ void k_bonded(Model m, Topo t, const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                         const int *__restrict__ orig,
                         const int *__restrict__ sorted_of, const float4 *__restrict__ add,
                         float4 *__restrict__ out_sum, float4 *__restrict__ out_bond) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const int o = orig[i];
    const D3 xi = full_pos(xs, xl, i);
    double gx = 0., gy = 0., gz = 0., en = 0.;
    for (int b = t.bptr[o]; b < t.bptr[o + 1]; ++b) {
        D3 xj = full_pos(xs, xl, sorted_of[t.bother[b]]);
        double dx = min_image_d(xi.x, xj.x, m.box[0]);
        double dy = min_image_d(xi.y, xj.y, m.box[1]);
        double dz = min_image_d(xi.z, xj.z, m.box[2]);
        double r = sqrt(dx * dx + dy * dy + dz * dz), dr = r - (double)t.br0[b], k = (double)t.bk[b];
        double f = 2.0 * k * dr / r;
        gx += f * dx; gy += f * dy; gz += f * dz;
        en += 0.5 * k * dr * dr;
    }
    for (int a = t.aptr[o]; a < t.aptr[o + 1]; ++a) {
        // role 1: I am the vertex, (aa, ab) are the ends; else I am an end, aa = vertex, ab = other end
        const int role = t.arole[a];
        D3 xa = full_pos(xs, xl, sorted_of[t.aa[a]]), xb = full_pos(xs, xl, sorted_of[t.ab[a]]);
        D3 xv = role == 1 ? xi : xa;             // vertex
        D3 xe1 = role == 1 ? xa : xi;            // end whose gradient is "gi"
        D3 xe2 = xb;                             // other end
        double u[3], w[3];
        u[0] = min_image_d(xe1.x, xv.x, m.box[0]);
        u[1] = min_image_d(xe1.y, xv.y, m.box[1]);
        u[2] = min_image_d(xe1.z, xv.z, m.box[2]);
        w[0] = min_image_d(xe2.x, xv.x, m.box[0]);
        w[1] = min_image_d(xe2.y, xv.y, m.box[1]);
        w[2] = min_image_d(xe2.z, xv.z, m.box[2]);
        double lu = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]), lw = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
        double ct = (u[0] * w[0] + u[1] * w[1] + u[2] * w[2]) / (lu * lw);
        ct = fmin(1.0, fmax(-1.0, ct));
        double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12);
        double dth = th - (double)t.at0[a], k = (double)t.ak[a], dU = 2.0 * k * dth;
        double g[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double gi = -dU * (w[c] / lw - ct * u[c] / lu) / (lu * st);
            if (role == 1) {
                double gk = -dU * (u[c] / lu - ct * w[c] / lw) / (lw * st);
                g[c] = -(gi + gk);
            } else g[c] = gi;
        }
        gx += g[0]; gy += g[1]; gz += g[2];
        en += k * dth * dth * (1.0 / 3.0);
    }
    float4 fb = make_float4((float)gx, (float)gy, (float)gz, (float)en);
    if (out_bond) out_bond[i] = fb;
    if (out_sum) {
        if (add) { float4 p = add[i]; fb.x += p.x; fb.y += p.y; fb.z += p.z; fb.w += p.w; }
        out_sum[i] = fb;
    }
}

// The same bonded terms with BONDED_LANES lanes per atom (lane l takes the terms l, l + BONDED_LANES, ... of the
// atom's bond-then-angle list; the partial sums are combined by shuffles in a fixed order: deterministic).
constexpr int BONDED_LANES = 4;
__device__ inline void bonded_term(const Model &m, const Topo &t, const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                   const int *__restrict__ sorted_of, int o, const D3 &xi, int term, int nb, double &gx,
                                   double &gy, double &gz, double &en) {
    if (term < nb) {
        const int b = t.bptr[o] + term;
        D3 xj = full_pos(xs, xl, sorted_of[t.bother[b]]);
        double dx = min_image_d(xi.x, xj.x, m.box[0]);
        double dy = min_image_d(xi.y, xj.y, m.box[1]);
        double dz = min_image_d(xi.z, xj.z, m.box[2]);
        double r = sqrt(dx * dx + dy * dy + dz * dz), dr = r - (double)t.br0[b], k = (double)t.bk[b];
        double f = 2.0 * k * dr / r;
        gx += f * dx; gy += f * dy; gz += f * dz;
        en += 0.5 * k * dr * dr;
        return;
    }
    const int a = t.aptr[o] + (term - nb);
    const int role = t.arole[a];
    D3 xa = full_pos(xs, xl, sorted_of[t.aa[a]]), xb = full_pos(xs, xl, sorted_of[t.ab[a]]);
    D3 xv = role == 1 ? xi : xa;
    D3 xe1 = role == 1 ? xa : xi;
    D3 xe2 = xb;
    double u[3], w[3];
    u[0] = min_image_d(xe1.x, xv.x, m.box[0]);
    u[1] = min_image_d(xe1.y, xv.y, m.box[1]);
    u[2] = min_image_d(xe1.z, xv.z, m.box[2]);
    w[0] = min_image_d(xe2.x, xv.x, m.box[0]);
    w[1] = min_image_d(xe2.y, xv.y, m.box[1]);
    w[2] = min_image_d(xe2.z, xv.z, m.box[2]);
    double lu = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]), lw = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
    double ct = (u[0] * w[0] + u[1] * w[1] + u[2] * w[2]) / (lu * lw);
    ct = fmin(1.0, fmax(-1.0, ct));
    double th = acos(ct), st = fmax(sqrt(1.0 - ct * ct), 1e-12);
    double dth = th - (double)t.at0[a], k = (double)t.ak[a], dU = 2.0 * k * dth;
    double g[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double gi = -dU * (w[c] / lw - ct * u[c] / lu) / (lu * st);
        if (role == 1) {
            double gk = -dU * (u[c] / lu - ct * w[c] / lw) / (lw * st);
            g[c] = -(gi + gk);
        } else g[c] = gi;
    }
    gx += g[0]; gy += g[1]; gz += g[2];
    en += k * dth * dth * (1.0 / 3.0);
}
__device__ inline void bonded_lanes(const Model &m, const Topo &t, const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                    const int *__restrict__ orig, const int *__restrict__ sorted_of,
                                    float4 *__restrict__ out_bond, int i, int gl, unsigned gmask) {
    double gx = 0., gy = 0., gz = 0., en = 0.;
    if (i < m.n) {
        const int o = orig[i];
        const D3 xi = full_pos(xs, xl, i);
        const int nb = t.bptr[o + 1] - t.bptr[o], nt = nb + t.aptr[o + 1] - t.aptr[o];
        for (int term = gl; term < nt; term += BONDED_LANES) bonded_term(m, t, xs, xl, sorted_of, o, xi, term, nb, gx, gy, gz, en);
    }
#pragma unroll
    for (int off = 1; off < BONDED_LANES; off <<= 1) {
        gx += __shfl_xor_sync(gmask, gx, off);
        gy += __shfl_xor_sync(gmask, gy, off);
        gz += __shfl_xor_sync(gmask, gz, off);
        en += __shfl_xor_sync(gmask, en, off);
    }
    if (gl == 0 && i < m.n) out_bond[i] = make_float4((float)gx, (float)gy, (float)gz, (float)en);
}

// bonded gradient alone, BONDED_LANES lanes per atom (a fused pair + bonded launch was tried: the fp64 bonded code
// raises the register count of the whole kernel and halves the occupancy of the pair warps -- 32 us instead of 20 + 4)
__global__ void __launch_bounds__(128) k_bonded_lanes(Model m, Topo t, const float4 *__restrict__ xs,
                                                      const float4 *__restrict__ xl, const int *__restrict__ orig,
                                                      const int *__restrict__ sorted_of, float4 *__restrict__ out_bond) {
    const int gt = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    const int i = gt / BONDED_LANES, gl = gt % BONDED_LANES;
    const unsigned gmask = ((1u << BONDED_LANES) - 1u) << (lane & ~(BONDED_LANES - 1));
    bonded_lanes(m, t, xs, xl, orig, sorted_of, out_bond, i, gl, gmask);
}

// out[orig[i]] = f[i].xyz  (sorted -> caller order)
__global__ void k_unsort3(int n, const float4 *__restrict__ f, const int *__restrict__ orig, float *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = f[i];
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
        float4 xj = xs[ridx[k]];
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
    const int B = 256;
    unsigned grid = (unsigned)(((long long)m.n * 32 + B - 1) / B);
    if (energy) k_pair<WC, WLJ, true><<<grid, B, 0, st>>>(m, row, xs, lj, out, accumulate);
    else k_pair<WC, WLJ, false><<<grid, B, 0, st>>>(m, row, xs, lj, out, accumulate);
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

void launch_bonded_lanes(const Model &m, const Topo &t, const float4 *xs, const float4 *xl, const int *orig,
                         const int *sorted_of, float4 *out_bond, cudaStream_t st, int64_t *launches) {
    const int B = 128;
    k_bonded_lanes<<<(unsigned)(((long long)m.n * BONDED_LANES + B - 1) / B), B, 0, st>>>(m, t, xs, xl, orig, sorted_of, out_bond);
    *launches += 1;
}

void launch_bonded(const Model &m, const Topo &t, const float4 *xs, const float4 *xl, const int *orig, const int *sorted_of,
                   const float4 *add, float4 *out_sum, float4 *out_bond, cudaStream_t st, int64_t *launches) {
    const int B = 128;
    k_bonded<<<(m.n + B - 1) / B, B, 0, st>>>(m, t, xs, xl, orig, sorted_of, add, out_sum, out_bond);
    *launches += 1;
}

void launch_unsort3(int n, const float4 *f, const int *orig, float *out, cudaStream_t st, int64_t *launches) {
    const int B = 256;
    k_unsort3<<<(n + B - 1) / B, B, 0, st>>>(n, f, orig, out);
    *launches += 1;
}

}  // namespace jb
