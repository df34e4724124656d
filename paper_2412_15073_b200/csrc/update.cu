// update.cu -- velocity half-phases (B kick / jump chains C', J') and the fused A-O-A drift
// (SURVEY 8(a) a6, a7, a8).
//
// C' : Algorithm 4 with the ring technique, as reconstructed in R-11.
// J' : Algorithm 5, BPS on the long LJ part, with an exponential clock (R-14).
// A, O: x += (delta/2) v;  v <- c1 v + c2 m^-1/2 G.
// Chains of different atoms are independent and a jump of type (i,j) changes v_i only
// (P:L342): one chain per thread, writing nothing but its own v_i -- no cross-atom conflict; several
// events on one atom are resolved in time order inside its chain.
#include <cstdlib>

#include "launch.h"

namespace jb {

struct Tally {  // per-thread statistics, reduced once per warp at the end
    unsigned proposals, accepts, gt_attempts, expiries;
    float max_p, max_gl;
};

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

// Theta(eta) = E[(eta+G)_+] = eta Phi(eta) + phi(eta)  (R-5)
__device__ inline float theta_of(float eta) {
    float Phi = 0.5f * erfcf(-eta * 0.70710678118654752f);
    float phi = kInvSqrt2Pi * expf(-0.5f * eta * eta);
    return eta * Phi + phi;
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

// long part of the Coulomb pair gradient, F_ij = grad_{x_i} (1-chi) u_C: returns fr = radial
// derivative, d = minimum-image x_i - x_j, r
__device__ inline float fij_coul(const Model &m, const float4 &xi, const float4 &xj, float &dx, float &dy, float &dz,
                                 float &rinv) {
    float ax, ay, az, bx, by, bz;
    image_pair1(xi.x, xj.x, m.box[0], m.inv_box[0], ax, bx);
    image_pair1(xi.y, xj.y, m.box[1], m.inv_box[1], ay, by);
    image_pair1(xi.z, xj.z, m.box[2], m.inv_box[2], az, bz);
    dx = ax - bx; dy = ay - by; dz = az - bz;
    float r2 = dx * dx + dy * dy + dz * dz;
    if (r2 >= m.rE2 || r2 <= m.rlo2) { rinv = 0.f; return 0.f; }
    rinv = rsqrtf(r2);
    float r = r2 * rinv;
    float qq = (float)kCoulomb * xi.w * xj.w;
    float ex = expf(-m.alpha2 * r2), e = ex * erfcx_poly(m.alpha * r);
    float u = qq * e * rinv;
    float du = -(u + qq * kTwoOverSqrtPi * m.alpha * ex) * rinv;
    float dchi, chi = chi_zone(ax, ay, az, bx, by, bz, r2, r, m, dchi);
    return (1.f - chi) * du - dchi * u;
}
__device__ inline float fij_lj(const Model &m, const float4 &xi, const float4 &xj, float2 lji, float2 ljj, float &dx,
                               float &dy, float &dz, float &rinv) {
    float ax, ay, az, bx, by, bz;
    image_pair1(xi.x, xj.x, m.box[0], m.inv_box[0], ax, bx);
    image_pair1(xi.y, xj.y, m.box[1], m.inv_box[1], ay, by);
    image_pair1(xi.z, xj.z, m.box[2], m.inv_box[2], az, bz);
    dx = ax - bx; dy = ay - by; dz = az - bz;
    float r2 = dx * dx + dy * dy + dz * dz;
    if (r2 >= m.rE2 || r2 <= m.rlo2) { rinv = 0.f; return 0.f; }
    rinv = rsqrtf(r2);
    float r = r2 * rinv;
    float s = lji.x * ljj.x * rinv, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
    float e4 = lji.y * ljj.y;
    float u = e4 * (s12 - s6), du = e4 * (6.f * s6 - 12.f * s12) * rinv;
    float dchi, chi = chi_zone(ax, ay, az, bx, by, bz, r2, r, m, dchi);
    return (1.f - chi) * du - dchi * u;
}

// ---- step (C'): Algorithm 4 + ring (R-11).  x frozen; updates (vx,vy,vz) of atom i. -------------------------
// G lanes cooperate on one chain.  What a proposal needs from the random stream and from x -- the exponential
// E, the ring, the partner j, the uniform U and the pair gradient F_ij(x) (x is frozen) -- does not depend on
// the chain's state (t, v), so lane l evaluates all of that for the l-th next iteration at once (Philox block
// b + l, the row and position gathers, erfc/exp).  Only the thinning recurrence itself is sequential
// (B_v -> lambda-bar -> T -> t, v -> accept test); every lane of the group replays it on the
// broadcast values, so (t, v) stay replicated in registers.  An accepted jump consumes G~ blocks and thereby
// shifts the block index of the later iterations (R-15): the speculative tail is then dropped and the batch
// restarted -- accepted jumps are ~1 % of the proposals.  The arithmetic of every iteration is exactly the
// sequential algorithm's, so the event log equals the oracle's whatever G is.
template <int G, bool LOG>
__device__ void chain_C(const Model &m, const UpdateArgs &A, int i, unsigned atom, const float4 &xi, float sbm,
                        float ax, float ay, float az, float H, unsigned stream, unsigned step, float &vx, float &vy,
                        float &vz, Tally &tl, unsigned gmask, int gl) {
    const float eps = m.eps_jump, beta = m.beta;
    const bool bps = isinf(eps);
    const int NM = A.rowM.cnt[i], NL = A.rowL.cnt[i];
    const float aq = fabsf(xi.w);
    const float LM = aq * m.qmaxGM, LL = aq * m.qmaxGL;
    const float SM = (float)NM * LM, S = SM + (float)NL * LL;
    const float lam0 = bps ? 0.f : (1.f / eps) * beta * kInvSqrt2Pi / sbm;
    const float a2 = ax * ax + ay * ay + az * az;
    const bool lead = gl == 0;
    float t = 0.f;
    unsigned block = 0;
    int iter = 0;
    if (!(S > 0.f)) {  // no partner: lambda-bar = 0, the clock never rings
        vx += H * ax; vy += H * ay; vz += H * az;
        if (lead) {
            tl.expiries++;
            if (LOG) log_event(A, step, stream, atom, 0, -1, -1, 0, 0, INFINITY, 0.f, 0.f, 0.f);
        }
        return;
    }
    for (;;) {
        // ---- state-independent part of iteration (iter + gl), Philox block (block + gl) ----
        uint32_t w[4];
        philox4x32_10(atom, step, stream, block + (unsigned)gl, m.key0, m.key1, w);
        float E_ = -logf(u01(w[0]));
        int ring_ = (u01(w[1]) * S < SM) ? 0 : 1;  // ring pick
        if (ring_ == 0 && NM == 0) ring_ = 1;
        if (ring_ == 1 && NL == 0) ring_ = 0;
        const int cnt = ring_ == 0 ? NM : NL;
        const int k = (int)__umulhi(w[2], (unsigned)cnt);
        const int j_ = ring_ == 0 ? A.rowM.idx[(size_t)i * A.rowM.cap + k] : A.rowL.idx[(size_t)i * A.rowL.cap + k];
        const float U_ = u01(w[3]);
        float dx, dy, dz, rinv;
        float fr = fij_coul(m, xi, A.xs[j_], dx, dy, dz, rinv);
        float g_ = fabsf(fr);
        float sg = (fr > 0.f ? rinv : -rinv);  // n = F/|F|
        float nx_ = dx * sg, ny_ = dy * sg, nz_ = dz * sg;
        const float LY_ = ring_ == 0 ? LM : LL;
        float gl_ = g_ / LY_;
        int jo_ = LOG ? A.orig[j_] : 0;
        // ---- the thinning recurrence over the G staged iterations ----
        bool finished = false, restart = false;
#pragma unroll 1
        for (int l = 0; l < G; ++l) {
            float E = __shfl_sync(gmask, E_, l, G);
            float tau = H - t;
            float va = vx * ax + vy * ay + vz * az;
            float v2 = vx * vx + vy * vy + vz * vz;
            float Bv = sqrtf(v2 + tau * tau * a2 + 2.f * tau * fmaxf(va, 0.f));
            float lam = S * (beta * Bv + lam0);
            float T = E / lam;   // P:L379 (lam = 0: +inf).  IEEE sqrt and division: t + T <= H is a fragile decision (R-17)
            if (!(t + T <= H)) {
                vx += tau * ax; vy += tau * ay; vz += tau * az;
                if (lead) {
                    tl.expiries++;
                    if (LOG) log_event(A, step, stream, atom, iter, -1, -1, 0, 0, T, 0.f, 0.f, 0.f);
                }
                finished = true;
                break;
            }
            t += T;
            vx += T * ax; vy += T * ay; vz += T * az;
            float g = __shfl_sync(gmask, g_, l, G), goL = __shfl_sync(gmask, gl_, l, G), U = __shfl_sync(gmask, U_, l, G);
            if (lead) { tl.proposals++; tl.max_gl = fmaxf(tl.max_gl, goL); }
            float p = 0.f, gt = 0.f;
            int acc = 0, att = 0;
            // p <= g / L_Y always (Theta(eta) <= eta_+ + 1/sqrt(2 pi), eta <= eps sqrt(beta m) B_v): most proposals
            // are rejected on that bound alone; p itself is evaluated when it can matter (or is logged)
            if (g > 0.f && (LOG || U <= goL * 1.0001f)) {
                float nx = __shfl_sync(gmask, nx_, l, G), ny = __shfl_sync(gmask, ny_, l, G), nz = __shfl_sync(gmask, nz_, l, G);
                float LY = __shfl_sync(gmask, LY_, l, G);
                float vn = vx * nx + vy * ny + vz * nz;
                if (bps) p = fmaxf(vn, 0.f) * g / (LY * Bv);
                else p = g * theta_of(eps * sbm * vn) / (LY * (Bv * eps * sbm + kInvSqrt2Pi));  // P:L397 with sqrt(beta)
                if (lead) tl.max_p = fmaxf(tl.max_p, p);
                if (U <= p) {
                    unsigned b2 = block + (unsigned)l + 1u;
                    if (!bps) gt = gtilde(eps * sbm * vn, atom, step, stream, b2, m, att);
                    jump_kick(eps, sbm, nx, ny, nz, gt, vx, vy, vz);
                    acc = 1;
                    if (lead) { tl.accepts++; tl.gt_attempts += att; }
                    block = b2;  // the next iteration's block follows the sampler's
                    restart = true;
                }
            }
            if (LOG) {
                int ring = __shfl_sync(gmask, ring_, l, G), jo = __shfl_sync(gmask, jo_, l, G);
                if (lead) log_event(A, step, stream, atom, iter, ring, jo, acc, att, T, p, U, gt);
            }
            ++iter;
            if (restart) break;
        }
        if (finished) break;
        if (!restart) block += (unsigned)G;
    }
}

// ---- step (J'): Algorithm 5 (R-14) ---------------------------------------------------------------------------
// Rare (LJ carriers only, ~0.15 proposals per fs): every lane of the group runs the same sequential chain.
__device__ void chain_J(const Model &m, const UpdateArgs &A, int i, unsigned atom, const float4 &xi, float2 lji,
                        float sbm, float H, unsigned stream, unsigned step, float &vx, float &vy, float &vz, Tally &tl,
                        bool lead) {
    if (!(lji.y > 0.f)) return;
    const int NV = A.rowV.cnt[i];
    if (NV == 0) return;
    const float L = 0.5f * lji.y * m.GV4se;  // 4 sqrt(eps_i eps_max) G_V; lji.y = 2 sqrt(eps_i)
    float t = 0.f;
    unsigned block = 0;
    uint32_t w[4];
    for (int iter = 0;; ++iter) {
        float vv = sqrtf(vx * vx + vy * vy + vz * vz);
        float lam = (float)NV * m.beta * vv * L;
        philox4x32_10(atom, step, stream, block++, m.key0, m.key1, w);
        float E = -logf(u01(w[0]));
        float T = lam > 0.f ? E / lam : INFINITY;
        if (!(t + T <= H)) {
            if (lead) {
                tl.expiries++;
                log_event(A, step, stream, atom, iter, -1, -1, 0, 0, T, 0.f, 0.f, 0.f);
            }
            break;
        }
        t += T;
        const int k = (int)__umulhi(w[1], (unsigned)NV);
        const int j = A.rowV.idx[(size_t)i * A.rowV.cap + k];
        const float U = u01(w[2]);
        if (lead) tl.proposals++;
        float dx, dy, dz, rinv;
        float fr = fij_lj(m, xi, A.xs[j], lji, A.lj[j], dx, dy, dz, rinv);
        float g = fabsf(fr), p = 0.f;
        int acc = 0;
        if (g > 0.f) {
            float sg = (fr > 0.f ? rinv : -rinv);
            float nx = dx * sg, ny = dy * sg, nz = dz * sg;
            float vF = (vx * nx + vy * ny + vz * nz) * g;
            p = fmaxf(vF, 0.f) / (vv * L);
            if (lead) { tl.max_gl = fmaxf(tl.max_gl, g / L); tl.max_p = fmaxf(tl.max_p, p); }
            if (U <= p) {  // reflection (5)
                jump_kick(INFINITY, sbm, nx, ny, nz, 0.f, vx, vy, vz);
                acc = 1;
                if (lead) tl.accepts++;
            }
        }
        if (lead) log_event(A, step, stream, atom, iter, 2, A.orig[j], acc, 0, T, p, U, 0.f);
    }
}

__device__ inline double wrap1d(double x, double L) {
    x -= L * floor(x / L);
    if (x >= L) x -= L;
    if (x < 0.0) x = 0.0;
    return x;
}

// ---- the fused per-atom update: up to two velocity half-phases, then A O A + wrap ----------------------------
// G lanes per atom (a power of two <= 32): they share the jump chains (see chain_C); lane 0 of the group does the
// A-O-A part and all the stores.
template <bool JUMPS, int G, bool LOG>
__global__ void __launch_bounds__(128) k_update(Model m, UpdateArgs A) {
    const unsigned full = 0xffffffffu;
    const int gt_id = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = gt_id / G, gl = gt_id % G;
    const int lane = threadIdx.x & 31;
    const unsigned gmask = (G == 32) ? full : (((1u << G) - 1u) << (lane & ~(G - 1)));
    const bool live = i < m.n, lead = gl == 0;
    Tally tl = {0u, 0u, 0u, 0u, 0.f, 0.f};
    float disp2 = 0.f;
    bool bad = false;
    if (live) {
        const float4 xi = A.xs[i];
        float4 v4 = A.vs[i];
        float vx = v4.x, vy = v4.y, vz = v4.z;
        const float2 mi = A.mi[i];  // (kcal-scaled 1/m, sqrt(beta m))
        const unsigned atom = (unsigned)A.orig[i];
#pragma unroll
        for (int ph = 0; ph < 2; ++ph) {
            const Phase &P = A.ph[ph];
            if (P.kind == 0) continue;
            float ax = 0.f, ay = 0.f, az = 0.f;
            if (P.use_grad) {  // a = -M^-1 F
                float4 g = A.grad[ph][i];
                if (A.grad_b[ph]) { float4 b = A.grad_b[ph][i]; g.x = b.x + g.x; g.y = b.y + g.y; g.z = b.z + g.z; }
                ax = -mi.x * g.x; ay = -mi.x * g.y; az = -mi.x * g.z;
            }
            if (P.kind == 1 || !JUMPS) {
                vx += P.H * ax; vy += P.H * ay; vz += P.H * az;
            } else {
                const float2 lji = A.lj[i];
                if (P.reverse && P.lj) chain_J(m, A, i, atom, xi, lji, mi.y, P.H, P.streamJ, P.step, vx, vy, vz, tl, lead);
                if (P.coul) chain_C<G, LOG>(m, A, i, atom, xi, mi.y, ax, ay, az, P.H, P.streamC, P.step, vx, vy, vz, tl, gmask, gl);
                else if (P.use_grad) { vx += P.H * ax; vy += P.H * ay; vz += P.H * az; }
                if (!P.reverse && P.lj) chain_J(m, A, i, atom, xi, lji, mi.y, P.H, P.streamJ, P.step, vx, vy, vz, tl, lead);
            }
        }
        if (A.do_aoa && lead) {
            // positions are integrated in fp64 as hi + lo (hi = the fp32 value every pair kernel reads):
            // fp32 rounding of x (ulp(18 A) = 2e-6 A) through the stiff O-H bonds is otherwise the
            // largest noise source of the whole step
            const float4 xlo = A.xl[i];
            double X = (double)xi.x + (double)xlo.x, Y = (double)xi.y + (double)xlo.y, Z = (double)xi.z + (double)xlo.z;
            const double hdt = (double)A.half_dt;
            X += hdt * (double)vx; Y += hdt * (double)vy; Z += hdt * (double)vz;  // A
            uint32_t w[4];                                                          // O
            philox4x32_10(atom, A.o_step, 0u, 0u, m.key0, m.key1, w);
            float r1 = sqrtf(-2.f * logf(u01(w[0]))), r2 = sqrtf(-2.f * logf(u01(w[2])));
            float s1, c1, c2;
            sincospif(2.f * u01(w[1]), &s1, &c1);
            c2 = cospif(2.f * u01(w[3]));
            float sc = A.c2 / mi.y;
            vx = A.c1 * vx + sc * (r1 * c1);
            vy = A.c1 * vy + sc * (r1 * s1);
            vz = A.c1 * vz + sc * (r2 * c2);
            X += hdt * (double)vx; Y += hdt * (double)vy; Z += hdt * (double)vz;  // A
            X = wrap1d(X, (double)m.box[0]); Y = wrap1d(Y, (double)m.box[1]); Z = wrap1d(Z, (double)m.box[2]);
            const float x = (float)X, y = (float)Y, z = (float)Z;
            A.xs_out[i] = make_float4(x, y, z, xi.w);
            A.xl[i] = make_float4((float)(X - (double)x), (float)(Y - (double)y), (float)(Z - (double)z), 0.f);
            float4 xb = A.x_build[i];
            float ddx = min_image1(x, xb.x, m.box[0], m.inv_box[0]);
            float ddy = min_image1(y, xb.y, m.box[1], m.inv_box[1]);
            float ddz = min_image1(z, xb.z, m.box[2], m.inv_box[2]);
            disp2 = ddx * ddx + ddy * ddy + ddz * ddz;
            bad = !(isfinite(x) && isfinite(y) && isfinite(z));
        }
        bad = bad || !(isfinite(vx) && isfinite(vy) && isfinite(vz));
        if (lead) A.vs[i] = make_float4(vx, vy, vz, v4.w);
    }
    // warp-level reduction of the statistics, then a few integer atomics per warp
    unsigned err = 0;
    if (bad) err |= ERR_NAN;
    if (disp2 > m.half_skin2) err |= ERR_SKIN;
    if (tl.max_p > 1.f + 1e-4f || tl.max_gl > 1.f + 1e-4f) err |= ERR_BOUND;
    unsigned d2b = __reduce_max_sync(full, __float_as_uint(disp2));
    err = __reduce_or_sync(full, err);
    if (JUMPS) {
        unsigned np = __reduce_add_sync(full, tl.proposals), na = __reduce_add_sync(full, tl.accepts);
        unsigned ng = __reduce_add_sync(full, tl.gt_attempts), ne = __reduce_add_sync(full, tl.expiries);
        unsigned mp = __reduce_max_sync(full, __float_as_uint(tl.max_p));
        unsigned mg = __reduce_max_sync(full, __float_as_uint(tl.max_gl));
        if (lane == 0) {
            if (np) atomicAdd(&A.ctr->proposals, (unsigned long long)np);
            if (na) atomicAdd(&A.ctr->accepts, (unsigned long long)na);
            if (ng) atomicAdd(&A.ctr->gt_attempts, (unsigned long long)ng);
            if (ne) atomicAdd(&A.ctr->expiries, (unsigned long long)ne);
            if (mp > A.ctr->max_p_bits) atomicMax(&A.ctr->max_p_bits, mp);
            if (mg > A.ctr->max_gl_bits) atomicMax(&A.ctr->max_gl_bits, mg);
        }
    }
    if (lane == 0) {
        if (d2b > A.ctr->max_disp2_bits) atomicMax(&A.ctr->max_disp2_bits, d2b);
        if (err) atomicOr(&A.ctr->err, err);
    }
}

// caller arrays (original order, n x 3) <-> sorted float4
__global__ void k_writeback(int n, const float4 *__restrict__ xs, const float4 *__restrict__ vs,
                            const int *__restrict__ orig, float *__restrict__ pos, float *__restrict__ vel) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int o = orig[i];
    float4 x = xs[i], v = vs[i];
    pos[3 * o] = x.x; pos[3 * o + 1] = x.y; pos[3 * o + 2] = x.z;
    vel[3 * o] = v.x; vel[3 * o + 1] = v.y; vel[3 * o + 2] = v.z;
}

// original order in: wrap positions, pack (x, q), (v), (sqrt sigma, 2 sqrt eps), (kcal/m, sqrt(beta m))
__global__ void k_load(Model m, const float *__restrict__ pos, const float *__restrict__ vel,
                       const float *__restrict__ mass, const float *__restrict__ charge,
                       const float *__restrict__ sigma, const float *__restrict__ eps, double kT, float4 *__restrict__ xs,
                       float4 *__restrict__ vs, float4 *__restrict__ xl, float2 *__restrict__ lj, float2 *__restrict__ mi,
                       int *__restrict__ orig) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    float x = wrap1(pos[3 * i], m.box[0], m.inv_box[0]);
    float y = wrap1(pos[3 * i + 1], m.box[1], m.inv_box[1]);
    float z = wrap1(pos[3 * i + 2], m.box[2], m.inv_box[2]);
    xs[i] = make_float4(x, y, z, charge[i]);
    vs[i] = make_float4(vel[3 * i], vel[3 * i + 1], vel[3 * i + 2], 0.f);
    xl[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    float e = eps[i];
    lj[i] = make_float2(e > 0.f ? (float)sqrt((double)sigma[i]) : 0.f, e > 0.f ? (float)(2.0 * sqrt((double)e)) : 0.f);
    double md = (double)mass[i];
    mi[i] = make_float2((float)(kKcal / md), (float)sqrt(md / (kT * kKcal)));
    orig[i] = i;
}

// re-read the caller's positions (wrapped) and velocities into the current sorted order
__global__ void k_reload(Model m, const float *__restrict__ pos, const float *__restrict__ vel,
                         const int *__restrict__ orig, float4 *__restrict__ xs, float4 *__restrict__ vs,
                         float4 *__restrict__ xl) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int o = orig[i];
    float4 x = xs[i];
    x.x = wrap1(pos[3 * o], m.box[0], m.inv_box[0]);
    x.y = wrap1(pos[3 * o + 1], m.box[1], m.inv_box[1]);
    x.z = wrap1(pos[3 * o + 2], m.box[2], m.inv_box[2]);
    xs[i] = x;
    xl[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    vs[i] = make_float4(vel[3 * o], vel[3 * o + 1], vel[3 * o + 2], 0.f);
}

// kinetic energy per atom into out[i] (kcal/mol), sorted order
__global__ void k_kinetic(int n, const float4 *__restrict__ vs, const float2 *__restrict__ mi, double *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = vs[i];
    double v2 = (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z;
    out[i] = 0.5 * v2 / (double)mi[i].x;  // (1/2) m v^2 / KCAL with mi.x = KCAL / m
}

template <int G>
static void update_dispatch(const Model &m, const UpdateArgs &A, bool jumps, cudaStream_t st) {
    const int B = 128;
    const unsigned grid = (unsigned)(((long long)m.n * G + B - 1) / B);
    if (!jumps) k_update<false, 1, false><<<(m.n + B - 1) / B, B, 0, st>>>(m, A);
    else if (A.events) k_update<true, G, true><<<grid, B, 0, st>>>(m, A);
    else k_update<true, G, false><<<grid, B, 0, st>>>(m, A);
}
// lanes per jump chain: as many as keep the grid within about two full waves of resident threads
// (148 SMs x 2048); JUMP_B200_LANES overrides (1, 4, 8, 16) for experiments
static int lanes_per_chain(int n) {
    static int forced = -1;
    if (forced < 0) {
        const char *e = getenv("JUMP_B200_LANES");
        forced = e ? atoi(e) : 0;
    }
    if (forced == 1 || forced == 4 || forced == 8 || forced == 16) return forced;
    const long long budget = 2ll * 148 * 2048;
    if ((long long)n * 16 <= budget) return 16;
    if ((long long)n * 8 <= budget) return 8;
    if ((long long)n * 4 <= budget) return 4;
    return 1;
}
void launch_update(const Model &m, const UpdateArgs &A, bool jumps, cudaStream_t st, int64_t *launches) {
    switch (jumps ? lanes_per_chain(m.n) : 1) {
        case 16: update_dispatch<16>(m, A, jumps, st); break;
        case 8: update_dispatch<8>(m, A, jumps, st); break;
        case 4: update_dispatch<4>(m, A, jumps, st); break;
        default: update_dispatch<1>(m, A, jumps, st); break;
    }
    *launches += 1;
}
void launch_writeback(int n, const float4 *xs, const float4 *vs, const int *orig, float *pos, float *vel, cudaStream_t st,
                      int64_t *launches) {
    k_writeback<<<(n + 255) / 256, 256, 0, st>>>(n, xs, vs, orig, pos, vel);
    *launches += 1;
}
void launch_load(const Model &m, const float *pos, const float *vel, const float *mass, const float *charge,
                 const float *sigma, const float *eps, double kT, float4 *xs, float4 *vs, float4 *xl, float2 *lj, float2 *mi,
                 int *orig, cudaStream_t st, int64_t *launches) {
    k_load<<<(m.n + 255) / 256, 256, 0, st>>>(m, pos, vel, mass, charge, sigma, eps, kT, xs, vs, xl, lj, mi, orig);
    *launches += 1;
}
void launch_reload(const Model &m, const float *pos, const float *vel, const int *orig, float4 *xs, float4 *vs,
                   float4 *xl, cudaStream_t st, int64_t *launches) {
    k_reload<<<(m.n + 255) / 256, 256, 0, st>>>(m, pos, vel, orig, xs, vs, xl);
    *launches += 1;
}
void launch_kinetic(int n, const float4 *vs, const float2 *mi, double *out, cudaStream_t st, int64_t *launches) {
    k_kinetic<<<(n + 255) / 256, 256, 0, st>>>(n, vs, mi, out);
    *launches += 1;
}

}  // namespace jb
