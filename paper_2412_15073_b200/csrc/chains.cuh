// chains.cuh -- device functions of the jump chains in the update kernel (update.cu): event log, Theta, the G~ sampler,
// the kick, single-pair long gradients, ring pick and candidate evaluation (
// R-5, R-6, R-10c).
#pragma once
#include "launch.h"

namespace jb {

struct Tally {  // per-thread statistics, reduced once per warp at the end
    unsigned proposals, accepts, gt_attempts, expiries;
    float max_p, max_gl;
    unsigned runaway;   // a chain was cut at kMaxChain proposals (reported as ERR_NAN: the state has blown up)
};
// A chain draws a few proposals per half-phase; with a non-finite or exploded velocity the bound lambda-bar is infinite,
// every waiting time is 0 and the clock never reaches the end of the phase: the chain is cut and the error flagged
// instead of spinning on the device for ever.
constexpr unsigned kMaxChain = 1u << 14;

__device__ inline void log_event(const UpdateArgs &a, unsigned step, int stream, int atom, int iter, int ring, int j,
                                 int accepted, int n_gt, float T, float p, float U, float gt) {
    if (!a.events) return;
    unsigned long long slot = atomicAdd(&a.ctr->n_events, 1ull);
    if (slot >= (unsigned long long)a.event_cap) { atomicOr(&a.ctr->err, (unsigned)ERR_EVENTS); return; }
    jump_event e;
    e.step = (int)step; e.stream = stream; e.atom = atom; e.iter = iter;
    e.ring = ring; e.j = j; e.accepted = accepted; e.n_gt = n_gt;
    e.T = T; e.p = p; e.U = U; e.gt = gt;
    a.events[slot] = e;
}

// Theta(eta) = E[(eta+G)_+] = eta Phi(eta) + phi(eta)  (R-5).  With x = |eta| / sqrt 2 both terms share
// e^{-x^2}: erfc(x) = e^{-x^2} erfcx_poly(x), phi = e^{-x^2} / sqrt(2 pi).  Beyond the polynomial's range
// (|eta| > 6.08) Theta is eta_+ to 1e-10, far below the smallest uniform (2^-24).
__device__ inline float theta_of(float eta) {
    const float x = fabsf(eta) * 0.70710678118654752f;
    if (x > 4.3f) return fmaxf(eta, 0.f);
    const float ex = expf(-x * x);
    const float half_erfc = 0.5f * ex * erfcx_poly(x);            // Phi(-|eta|)
    const float Phi = eta > 0.f ? 1.f - half_erfc : half_erfc;
    return fmaf(eta, Phi, kInvSqrt2Pi * ex);
}

// G~ ~ f_eta by rejection (R-6; proposal family of P:L310).  One Philox block per attempt.
__device__ inline float gtilde(float eta, unsigned atom, unsigned step, unsigned stream, unsigned &block,
                               const Model &m, int &attempts) {
    uint32_t w[4];
    int it = 0;
    float out = 0.f;
    for (;;) {
        ++it;
        philox4x32_10(atom, step, stream, block++, m.key0, m.key1, w);
        float u0 = u01(w[0]), u1 = u01(w[1]), u2 = u01(w[2]), u3 = u01(w[3]);
        if (eta < -2.5f) {  // Gamma(2, |eta|)
            float z = -(logf(u0) + logf(u1)) / fabsf(eta);
            if (u2 <= expf(-0.5f * z * z)) { out = z - eta; break; }
        } else if (eta < -1.f) {  // Exponential(|eta|)
            float z = -logf(u0) / fabsf(eta);
            if (u1 <= z * expf(0.5f * (1.f - z * z))) { out = z - eta; break; }
        } else if (eta <= 0.f) {  // Rayleigh
            float z = sqrtf(-2.f * logf(u0));
            if (u1 <= expf(eta * z)) { out = z - eta; break; }
        } else {  // Rayleigh-Gaussian mixture
            float wR = 1.f / (1.f + eta * kSqrt2Pi);
            if (u0 <= wR) { out = sqrtf(-2.f * logf(u1)); break; }
            float y = sqrtf(-2.f * logf(u1)) * cospif(2.f * u2);
            if (y > 0.f) { out = y; break; }
            if (y > -eta) {
                if (u3 <= (eta + y) / eta) { out = y; break; }
            }
        }
        if (it >= 64) { out = (eta > 0.f) ? 0.f : -eta + 1.f; break; }
    }
    attempts = it;
    return out;
}

// kick (7); eps = inf -> reflection (5)
__device__ inline void jump_kick(float eps, float sbm, float nx, float ny, float nz, float gt, float &vx, float &vy,
                                 float &vz) {
    float vn = vx * nx + vy * ny + vz * nz, amp;
    if (isinf(eps)) amp = 2.f * vn;
    else amp = 2.f * eps / ((1.f + eps * eps) * sbm) * (eps * sbm * vn + gt);
    vx -= amp * nx; vy -= amp * ny; vz -= amp * nz;
}

// geometry of a candidate pair: exact image pair (a, b) per dimension, d = a - b, r^2
struct PairGeom { float ax, ay, az, bx, by, bz, dx, dy, dz, r2; };
__device__ inline PairGeom pair_geom(const Model &m, const float4 &xi, const float4 &xj) {
    PairGeom p;
    image_pair1(xi.x, xj.x, m.box[0], m.inv_box[0], p.ax, p.bx);
    image_pair1(xi.y, xj.y, m.box[1], m.inv_box[1], p.ay, p.by);
    image_pair1(xi.z, xj.z, m.box[2], m.inv_box[2], p.az, p.bz);
    p.dx = p.ax - p.bx; p.dy = p.ay - p.by; p.dz = p.az - p.bz;
    p.r2 = p.dx * p.dx + p.dy * p.dy + p.dz * p.dz;
    return p;
}
// long part of the Coulomb pair gradient, F_ij = grad_{x_i} (1-chi) u_C: returns the radial derivative
__device__ inline float fij_coul(const Model &m, const PairGeom &p, float qi, float qj, float &rinv) {
    if (p.r2 >= m.rE2 || p.r2 <= m.rlo2) { rinv = 0.f; return 0.f; }
    rinv = rsqrtf(p.r2);
    float r = p.r2 * rinv;
    float qq = (float)kCoulomb * qi * qj;
    float ex = expf(-m.alpha2 * p.r2), e = ex * erfcx_poly(m.alpha * r);
    float u = qq * e * rinv;
    float du = -(u + qq * kTwoOverSqrtPi * m.alpha * ex) * rinv;
    float dchi, chi = chi_zone<true>(p.ax, p.ay, p.az, p.bx, p.by, p.bz, p.r2, r, m, dchi);
    return (1.f - chi) * du - dchi * u;
}
__device__ inline float fij_lj(const Model &m, const PairGeom &p, float2 lji, float2 ljj, float &rinv) {
    if (p.r2 >= m.rE2 || p.r2 <= m.rlo2 || !(ljj.y > 0.f)) { rinv = 0.f; return 0.f; }
    rinv = rsqrtf(p.r2);
    float r = p.r2 * rinv;
    float s = lji.x * ljj.x * rinv, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
    float e4 = lji.y * ljj.y;
    float u = e4 * (s12 - s6), du = e4 * (6.f * s6 - 12.f * s12) * rinv;
    float dchi, chi = chi_zone<true>(p.ax, p.ay, p.az, p.bx, p.by, p.bz, p.r2, r, m, dchi);
    return (1.f - chi) * du - dchi * u;
}

// ---- step (C'): Algorithm 4 + ring (R-11) --------------------------------------------------------------------
// G lanes cooperate on one chain, and nothing in the common case is sequential:
//  * what proposal k needs from the random stream and from x -- the exponential E_k, the ring, the partner j, the
//    uniform U_k and the pair gradient F_ij(x) -- depends neither on the chain's state nor on the other
//    proposals (x is frozen during a jump phase; proposal k draws Philox block k of its stream, the G~ attempts
//    have a stream of their own, R-15): lane l evaluates proposal kb + l;
//  * the bound lambda-bar is re-evaluated after each ACCEPTED jump only (R-11), so between two accepted
//    jumps the proposal times are a running sum of E_k / lambda-bar and v(t) = v_e + (t - t_e) a in closed form:
//    every lane gets its own proposal time (an inclusive scan over the group), its expiry test, its acceptance
//    probability and its accept test at once;
//  * the first accepting lane (a ballot) ends the epoch: kick, new bound, the later lanes are dropped and the
//    batch restarts after it -- accepted jumps are ~1-2 % of the proposals.
struct ChainConst {   // per-atom constants of the jump chains (R-10c): the three rings of P:L424
    int N[3];         // candidates: row A, row B, the cell universe of the home cell
    int home;         // home cell (ring C), packed coordinates
    bool far_excl;    // an excluded partner may be as far as ring C
};
__device__ inline ChainConst chain_const(const UpdateArgs &A, int i) {
    ChainConst c;
    c.N[0] = A.rowA.cnt[i]; c.N[1] = A.rowB.cnt[i];
    const int hp = A.uni.cell_of[i];   // bit 30: far-exclusion flag (sort_build.cu)
    c.home = hp & 0x3fffffff;
    c.far_excl = (hp >> 30) & 1;
    c.N[2] = universe_size(A.grid, A.uni, c.home);
    return c;
}
// N_Y by selects: an index computed at run time would put the three counts into local memory
__device__ __forceinline__ int ring_count(const ChainConst &c, int ring) { return ring == 0 ? c.N[0] : (ring == 1 ? c.N[1] : c.N[2]); }
// ring pick: the first ring whose cumulated weight exceeds ur * (sum of weights); a ring without
// candidates can only be hit through rounding at an end, and the pick then falls back as the oracle's does
__device__ inline int pick_ring(const ChainConst &c, float ur, float c0, float c1, float tot) {
    const float x = ur * tot;
    int ring = x < c0 ? 0 : (x < c1 ? 1 : 2);
    while (ring_count(c, ring) == 0 && ring > 0) --ring;
    while (ring_count(c, ring) == 0 && ring < 2) ++ring;
    return ring;
}
// A candidate j of ring `ring` (R-10c): the ring the pair's CURRENT distance lies in carries its force, through any
// other ring its rate is 0; then g = |F_ij| and n = F_ij / |F_ij|.  LJ: the long LJ gradient (step J') instead of the
// Coulomb one.  An fp32 r^2 within RING_TIE of a ring edge is re-decided in fp64 from the full positions (R-17).
// far_excl: the atom has an excluded partner that could be as far as ring C (never so in water): only then the
// universe's candidates are checked against the exclusion list (R-9).
// MODE 0: the long Coulomb gradient (step C'), 1: the long LJ gradient (step J'), 2: their sum (R-22)
template <int MODE>
__device__ inline void eval_candidate(const Model &m, const UpdateArgs &A, int ring, int i, int j, const float4 &xi, float2 lji,
                                      bool far_excl, float &g, float &nx, float &ny, float &nz) {
    const float4 xj = A.xs[j];
    const PairGeom p = pair_geom(m, xi, xj);
    const float lo2 = m.ring2[ring], hi2 = m.ring2[ring + 1];
    bool in = p.r2 >= lo2 && p.r2 < hi2;
    if (fminf(fabsf(p.r2 - lo2), fabsf(p.r2 - hi2)) < RING_TIE) {   // decide in fp64 from the full positions, like the oracle
        const float4 li = A.xl_all[i], lo_j = A.xl_all[j];
        double d[3] = {((double)xi.x + (double)li.x) - ((double)xj.x + (double)lo_j.x),
                       ((double)xi.y + (double)li.y) - ((double)xj.y + (double)lo_j.y),
                       ((double)xi.z + (double)li.z) - ((double)xj.z + (double)lo_j.z)};
        double r2d = 0.0;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const double L = (double)m.box[q];
            d[q] -= L * rint(d[q] / L);
            r2d += d[q] * d[q];
        }
        in = r2d >= m.ring2d[ring] && r2d < m.ring2d[ring + 1];
    }
    if (in && ring == 2 && far_excl) {   // the universe is not filtered at a build: excluded partners have rate 0 (R-9)
        const int o = A.orig[i], oj = A.orig[j];
        for (int e = A.excl_ptr[o]; e < A.excl_ptr[o + 1]; ++e) in = in && A.excl_idx[e] != oj;
    }
    float rinv = 0.f, fr = 0.f;
    if (in) fr = MODE == 1 ? fij_lj(m, p, lji, A.lj[j], rinv) : fij_coul(m, p, xi.w, xj.w, rinv);
    if (MODE == 2 && in) {   // R-22: F_ij is the whole long pair gradient (both parts lie along the pair axis)
        float rinv_lj;
        fr += fij_lj(m, p, lji, A.lj[j], rinv_lj);
    }
    const float sg = (fr > 0.f ? rinv : -rinv);  // n = F/|F|
    g = fabsf(fr);
    nx = p.dx * sg; ny = p.dy * sg; nz = p.dz * sg;
}
// candidate k of ring `ring` of atom i (home cell c.home): an entry of row A or B, or the k-th atom of the cell universe
__device__ inline int ring_candidate(const UpdateArgs &A, const ChainConst &c, int i, int ring, int k) {
    if (ring == 0) return A.rowA.idx[(size_t)i * A.rowA.cap + k];
    if (ring == 1) return A.rowB.idx[(size_t)i * A.rowB.cap + k];
    return universe_pick(A.grid, A.uni, A.cell_start, c.home, k);
}
// state-independent part of a proposal, from its Philox block w: ring pick and partner, then the pair;
// tag = ring << 28 | j_orig (event log only)
template <int MODE, bool WANT_J>
__device__ inline void propose_pair(const Model &m, const UpdateArgs &A, const ChainConst &c, float c0, float c1, float tot,
                                    int i, const float4 &xi, float2 lji, const uint32_t w[4], float &g, int &ring, float &nx,
                                    float &ny, float &nz, int &tag) {
    ring = pick_ring(c, u01(w[1]), c0, c1, tot);
    const int j = ring_candidate(A, c, i, ring, (int)__umulhi(w[2], (unsigned)ring_count(c, ring)));
    eval_candidate<MODE>(m, A, ring, i, j, xi, lji, c.far_excl, g, nx, ny, nz);
    tag = 0;
    if (WANT_J) tag = A.orig[j] | ((ring + (MODE == 2 ? 8 : 0)) << 28);   // ring codes 8-10: the combined mechanism
}

__device__ inline double wrap1d(double x, double L, double invL, int &img) {   // img += the number of box lengths taken off
    const double k = floor(x * invL);   // (a product, not the 40-instruction fp64 division; off by one at most, fixed below)
    x -= L * k;
    int ik = (int)k;
    if (x >= L) { x -= L; ++ik; }
    if (x < 0.0) { x += L; --ik; }
    if (x >= L || x < 0.0) x = 0.0;
    img += ik;
    return x;
}

}  // namespace jb
