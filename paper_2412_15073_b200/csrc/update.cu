// update.cu -- velocity half-phases (B kick / jump chains C', J') and the fused A-O-A drift
// (SURVEY 8(a) a6, a7, a8).
//
// C' : Algorithm 4 with the ring technique, as reconstructed in R-11.
// J' : Algorithm 5, BPS on the long LJ part, with an exponential clock (R-14).
// A, O: x += (delta/2) v;  v <- c1 v + c2 m^-1/2 G.
// Chains of different atoms are independent and a jump of type (i,j) changes v_i only
// (P:L342): one chain per thread, writing nothing but its own v_i -- no cross-atom conflict; several
// events on one atom are resolved in time order inside its chain.
#include "chains.cuh"

namespace jb {

// The chain of one atom, run by the G lanes of its group.  The whole warp executes the loop together (while any
// of its 32 / G groups still has a live chain, finished groups predicated off): groups of one warp never run one
// after the other, and every shuffle and ballot is a full-warp one.  `on` = this lane's atom exists and runs C'.
// ADAPT: eps(x) = eps0 |F_ij(x)| (R-19): per-pair bound beta L_Y B_v + lam0, p = Theta(eta) / (eps0
// sqrt(beta m) L_Y B_v + 1/sqrt(2 pi)), G~ and the kick (7) with eps = eps0 |F_ij|.
// MECH 0: constant eps; 1 (ADAPT): adaptive eps; 2 (COMB): constant eps on the whole long pair gradient, Coulomb + LJ (R-22)
template <int G, bool LOG, int MECH>
__device__ void chain_C(const Model &m, const UpdateArgs &A, bool on, const ChainConst &c, int i, unsigned atom, const float4 &xi,
                        float2 lji, float sbm, float ax, float ay, float az, float H, unsigned stream, unsigned step, float &vx, float &vy,
                        float &vz, Tally &tl, int gl, int gshift) {
    constexpr bool ADAPT = MECH == 1, COMB = MECH == 2;
    const unsigned full = 0xffffffffu;
    const float eps = m.eps_jump, beta = m.beta;
    const bool bps = isinf(eps), lead = gl == 0;
    const float aq = fabsf(xi.w);
    // L_Y,i = |q_i| q_max G_Y (R-7); combined mechanism (R-22): + sqrt(eps_i) 4 sqrt(eps_max) GV_Y, the LJ bound of the ring
    const float se = COMB ? 0.5f * lji.y : 0.f;
    const float L0 = fmaf(se, m.GV4se[0], aq * m.qmaxG[0]), L1 = fmaf(se, m.GV4se[1], aq * m.qmaxG[1]),
                L2 = fmaf(se, m.GV4se[2], aq * m.qmaxG[2]);
    const float w0 = (float)c.N[0] * L0, w1 = (float)c.N[1] * L1, w2 = (float)c.N[2] * L2;
    const float S = (w0 + w1) + w2;
    bool done = !(on && S > 0.f);
    if (on && done && lead) {  // no partner: lambda-bar = 0, the clock never rings; v drifts to the end below
        tl.expiries++;
        if (LOG) log_event(A, step, stream, atom, 0, -1, -1, 0, 0, INFINITY, 0.f, 0.f, 0.f);
    }
    const float lam0 = bps ? 0.f : (1.f / eps) * beta * kInvSqrt2Pi / sbm;
    const float a2 = ax * ax + ay * ay + az * az, esb = eps * sbm;
    const unsigned gbits = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    float vex = vx, vey = vy, vez = vz, te = 0.f;   // epoch start: velocity and time after the last accepted jump
    float t_run = 0.f;                              // time of the last proposal so far
    float Bv = 0.f, lam = 1.f, den = 1.f;
    float c0 = w0, c1 = w0 + w1, tot = S;   // ring Y is picked by ur * tot against the cumulated weights
    bool fresh = true;
    unsigned kb = 0, gblock = 0;
    while (__any_sync(full, !done)) {
        if (fresh) {   // the bound of this epoch, P:L373-374 (R-11: held until the next accepted jump)
            const float tau = H - te;
            const float va = vex * ax + vey * ay + vez * az, v2 = vex * vex + vey * vey + vez * vez;
            Bv = sqrtf(v2 + tau * tau * a2 + 2.f * tau * fmaxf(va, 0.f));
            if (ADAPT) {   // sum over the candidates of lambda*_Y (R-19)
                c0 = (float)c.N[0] * fmaf(beta * L0, Bv, lam0);
                c1 = c0 + (float)c.N[1] * fmaf(beta * L1, Bv, lam0);
                tot = c1 + (float)c.N[2] * fmaf(beta * L2, Bv, lam0);
                lam = tot;
            } else {
                lam = S * (beta * Bv + lam0);
                den = bps ? Bv : fmaf(Bv, esb, kInvSqrt2Pi);
            }
            fresh = false;
        }
        // lane gl draws Philox block kb + gl of the chain's stream: (E, ring, j, U) of proposal kb + gl (R-15)
        uint32_t w[4];
        philox4x32_10(atom, step, stream, kb + (unsigned)gl, m.key0, m.key1, w);
        const float T_ = done ? INFINITY : __fdividef(-logf(u01(w[0])), lam);   // P:L379 (lam = 0: +inf); 2-ulp division
        // time of my proposal: t_run + (T_0 + ... + T_gl), an inclusive scan over the group in log2 G shuffle steps
        // (the fp32 sum is associated differently from a sequential chain's: 1e-7 relative, far inside the
        // margins of R-17)
        float tk = T_;
#pragma unroll
        for (int off = 1; off < G; off <<= 1) {
            const float up = __shfl_up_sync(full, tk, off, G);
            if (gl >= off) tk += up;
        }
        tk += t_run;
        const bool alive = !done && tk <= H;   // the chain expires at the first proposal with t + T > delta/2
        const float U = u01(w[3]);
        float g = 0.f, nx = 0.f, ny = 0.f, nz = 0.f;
        int tag = 0, ring = 0;
        if (alive) propose_pair<COMB ? 2 : 0, LOG>(m, A, c, c0, c1, tot, i, xi, lji, w, g, ring, nx, ny, nz, tag);
        const float LY = ring == 0 ? L0 : (ring == 1 ? L1 : L2);
        const float goL = __fdividef(g, LY);
        float p = 0.f, vn = 0.f;
        bool acc = false;
        if (ADAPT) {
            if (alive && g > 0.f) {
                const float s = tk - te;
                const float cx = fmaf(s, ax, vex), cy = fmaf(s, ay, vey), cz = fmaf(s, az, vez);  // the advanced v
                vn = cx * nx + cy * ny + cz * nz;
                const float eta = esb * g * vn, dena = fmaf(esb * LY, Bv, kInvSqrt2Pi);            // esb = eps0 sqrt(beta m)
                if (LOG || U * dena <= (fmaxf(eta, 0.f) + kInvSqrt2Pi) * 1.0001f) {               // Theta <= eta_+ + 1/sqrt(2 pi)
                    p = theta_of(eta) / dena;
                    acc = U <= p;
                }
            }
        } else
        // p <= |F_ij| / L_Y always (Theta(eta) <= eta_+ + 1/sqrt(2 pi), eta <= eps sqrt(beta m) B_v): most proposals
        // are rejected on that bound alone; p itself is evaluated when it can matter (or is logged)
        if (alive && goL > 0.f && (LOG || U <= goL * 1.0001f)) {
            const float s = tk - te;
            const float cx = fmaf(s, ax, vex), cy = fmaf(s, ay, vey), cz = fmaf(s, az, vez);  // the advanced v
            vn = cx * nx + cy * ny + cz * nz;
            const float pub = bps ? goL * fmaxf(vn, 0.f) / den : goL * (fmaxf(esb * vn, 0.f) + kInvSqrt2Pi) / den;
            if (LOG || U <= pub * 1.0001f) {
                p = bps ? fmaxf(vn, 0.f) * goL / den : goL * theta_of(esb * vn) / den;  // P:L397 with sqrt(beta)
                acc = U <= p;
            }
        }
        // (G = 1: the group is the lane itself -- no ballots, no shuffles)
        const unsigned alive_m = G == 1 ? (alive ? 1u : 0u) : ((__ballot_sync(full, alive) >> gshift) & gbits);
        const unsigned acc_m = G == 1 ? (acc ? 1u : 0u) : ((__ballot_sync(full, acc) >> gshift) & gbits);
        const int n_alive = __popc(alive_m);
        const int f = acc_m ? __ffs(acc_m) - 1 : -1;   // first accepted proposal of the batch
        const int n_used = f >= 0 ? f + 1 : n_alive;
        const int fs = f >= 0 ? f : 0;
        const float tf = G == 1 ? tk : __shfl_sync(full, tk, fs, G), vnf = G == 1 ? vn : __shfl_sync(full, vn, fs, G);
        const float gf = ADAPT ? (G == 1 ? g : __shfl_sync(full, g, fs, G)) : 1.f;
        const float fnx = G == 1 ? nx : __shfl_sync(full, nx, fs, G), fny = G == 1 ? ny : __shfl_sync(full, ny, fs, G),
                    fnz = G == 1 ? nz : __shfl_sync(full, nz, fs, G);
        const float t_last = G == 1 ? tk : __shfl_sync(full, tk, G - 1, G);
        if (done) continue;
        if (gl < n_used) { tl.max_gl = fmaxf(tl.max_gl, goL); tl.max_p = fmaxf(tl.max_p, p); }
        if (lead) tl.proposals += (unsigned)n_used;
        float gt = 0.f;
        int att = 0;
        if (f >= 0) {   // kick (7) on the velocity at the time of proposal f; a new epoch starts there
            const float eps_ij = ADAPT ? eps * gf : eps;   // eps(x) = eps0 |F_ij(x)|
            if (!bps) gt = gtilde(eps_ij * sbm * vnf, atom, step, stream + 16u, gblock, m, att);
            const float s = tf - te;
            float cx = fmaf(s, ax, vex), cy = fmaf(s, ay, vey), cz = fmaf(s, az, vez);
            jump_kick(eps_ij, sbm, fnx, fny, fnz, gt, cx, cy, cz);
            vex = cx; vey = cy; vez = cz; te = tf; t_run = tf;
            fresh = true;
            if (lead) { tl.accepts++; tl.gt_attempts += att; }
        }
        if (LOG) {
            if (gl < n_used)
                log_event(A, step, stream, atom, (int)kb + gl, (int)((unsigned)tag >> 28), tag & 0x0fffffff, gl == f ? 1 : 0,
                          gl == f ? att : 0, T_, p, U, gl == f ? gt : 0.f);
            else if (f < 0 && gl == n_alive)
                log_event(A, step, stream, atom, (int)kb + gl, -1, -1, 0, 0, T_, 0.f, 0.f, 0.f);
        }
        if (kb > kMaxChain) { done = true; tl.runaway = 1u; }
        if (f >= 0) kb += (unsigned)(f + 1);
        else if (n_alive < G) {   // expired inside this batch
            done = true;
            if (lead) tl.expiries++;
        } else { t_run = t_last; kb += (unsigned)G; }
    }
    if (on) {   // drift to the end of the half-step
        const float s_end = H - te;
        vx = fmaf(s_end, ax, vex); vy = fmaf(s_end, ay, vey); vz = fmaf(s_end, az, vez);
    }
}

// ---- step (J'): Algorithm 5 (R-14), with the rings of R-10c ------------------------------------------------------
// Rare (LJ carriers only, ~0.1 proposals per fs): every lane of the group runs the same sequential chain.  The bound
// beta |v| sum_Y N_Y L^vdW_Y is constant over the half-step (|v| is preserved by reflections).
__device__ void chain_J(const Model &m, const UpdateArgs &A, const ChainConst &c, int i, unsigned atom, const float4 &xi,
                        float2 lji, float sbm, float H, unsigned stream, unsigned step, float &vx, float &vy, float &vz,
                        Tally &tl, bool lead) {
    if (!(lji.y > 0.f)) return;
    const float hs = 0.5f * lji.y;   // sqrt(eps_i); L^vdW_Y,i = 4 sqrt(eps_i eps_max) GV_Y
    const float L0 = hs * m.GV4se[0], L1 = hs * m.GV4se[1], L2 = hs * m.GV4se[2];
    const float w0 = (float)c.N[0] * L0, w1 = (float)c.N[1] * L1, w2 = (float)c.N[2] * L2;
    const float c0 = w0, c1 = w0 + w1, S = (w0 + w1) + w2;
    if (!(S > 0.f)) return;
    float t = 0.f;
    unsigned block = 0;
    uint32_t w[4];
    for (int iter = 0;; ++iter) {
        if ((unsigned)iter > kMaxChain) { tl.runaway = 1u; break; }
        float vv = sqrtf(vx * vx + vy * vy + vz * vz);
        float lam = S * (m.beta * vv);
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
        const float U = u01(w[3]);
        if (lead) tl.proposals++;
        float g, nx, ny, nz, p = 0.f;
        int ring, tag, acc = 0;
        propose_pair<1, true>(m, A, c, c0, c1, S, i, xi, lji, w, g, ring, nx, ny, nz, tag);
        const float L = ring == 0 ? L0 : (ring == 1 ? L1 : L2);
        if (g > 0.f) {
            float vF = (vx * nx + vy * ny + vz * nz) * g;
            p = fmaxf(vF, 0.f) / (vv * L);
            if (lead) { tl.max_gl = fmaxf(tl.max_gl, g / L); tl.max_p = fmaxf(tl.max_p, p); }
            if (U <= p) {  // reflection (5)
                jump_kick(INFINITY, sbm, nx, ny, nz, 0.f, vx, vy, vz);
                acc = 1;
                if (lead) tl.accepts++;
            }
        }
        if (lead) log_event(A, step, stream, atom, iter, 4 + ring, tag & 0x0fffffff, acc, 0, T, p, U, 0.f);
    }
}

// ---- the fused per-atom update: up to two velocity half-phases, then A O A + wrap ----------------------------
// G lanes per atom (a power of two <= 32) share the atom's jump chains; lane 0 of the group does A-O-A and the stores.
template <bool JUMPS, int G, bool LOG, int MECH>
__global__ void __launch_bounds__(128, 8) k_update(Model m, UpdateArgs A) {
    const unsigned full = 0xffffffffu;
    // a non-finite or blown-up state was flagged by an earlier launch: it is reported at the next synchronising call, and
    // until then the steps already enqueued do nothing (their chains would each run to the cut, 16 384 proposals)
    if (A.ctr->err & (unsigned)ERR_NAN) return;
    const int gt_id = blockIdx.x * blockDim.x + threadIdx.x;
    int i = gt_id / G;
    const int gl = gt_id % G;
    const int lane = threadIdx.x & 31, gshift = lane & ~(G - 1);
    if (JUMPS && G == 1) {
        // One chain per lane: a warp runs as long as its longest chain, and the chains of the strongly charged atoms
        // (rate ~ |q_i|: the oxygens of water, which also run the J' chains) are about twice as long as the others'.
        // The 128 atoms of the CTA are therefore dealt to its lanes with those atoms first (a stable partition): the
        // warps become homogeneous, and the ones with the short chains finish early.
        __shared__ int s_heavy[4];
        __shared__ unsigned char s_perm[128];
        const bool heavy = i < m.n && fabsf(A.xs[i].w) > m.q_split;
        const unsigned hb = __ballot_sync(full, heavy);
        const int wp = threadIdx.x >> 5;
        if (lane == 0) s_heavy[wp] = __popc(hb);
        __syncthreads();
        int before = __popc(hb & ((1u << lane) - 1u)), total = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { const int hk = s_heavy[k]; before += k < wp ? hk : 0; total += hk; }
        s_perm[heavy ? before : total + ((int)threadIdx.x - before)] = (unsigned char)threadIdx.x;
        __syncthreads();
        i = blockIdx.x * 128 + s_perm[threadIdx.x];
    }
    const bool live = i < m.n, lead = gl == 0;
    Tally tl = {0u, 0u, 0u, 0u, 0.f, 0.f, 0u};
    float disp2 = 0.f;
    bool bad = false;
    float4 xi = make_float4(0.f, 0.f, 0.f, 0.f), v4 = xi;
    float2 mi = make_float2(1.f, 1.f);   // (kcal-scaled 1/m, sqrt(beta m))
    unsigned atom = 0u;
    // everything the phases read from global memory is requested up front, in one batch of independent loads:
    // state, the accelerations of both phases, the ring counts (the per-phase dependent loads were a visible
    // part of a warp's latency chain)
    const bool jumpy0 = JUMPS && A.ph[0].kind == 2, jumpy1 = JUMPS && A.ph[1].kind == 2;
    const bool any_coul = (jumpy0 && A.ph[0].coul) || (jumpy1 && A.ph[1].coul);
    const bool any_lj = (jumpy0 && A.ph[0].lj) || (jumpy1 && A.ph[1].lj);
    float a0x = 0.f, a0y = 0.f, a0z = 0.f, a1x = 0.f, a1y = 0.f, a1z = 0.f;   // accelerations of the two phases
    ChainConst cc;
    cc.N[0] = cc.N[1] = cc.N[2] = 0; cc.home = 0; cc.far_excl = false;
    float2 lji = make_float2(0.f, 0.f);
    if (live) {
        xi = A.xs[i]; v4 = A.vs[i]; mi = A.mi[i]; atom = (unsigned)A.orig[i];
        const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 g0 = z4, g1 = z4, b0 = z4, b1 = z4;
        if (A.ph[0].kind != 0 && A.ph[0].use_grad) { g0 = A.grad[0][i]; if (A.grad_b[0]) b0 = A.grad_b[0][i]; }
        if (A.ph[1].kind != 0 && A.ph[1].use_grad) { g1 = A.grad[1][i]; if (A.grad_b[1]) b1 = A.grad_b[1][i]; }
        if (any_coul || any_lj) cc = chain_const(A, i);
        if (any_lj || MECH == 2) lji = A.lj[i];
        // a = -M^-1 F
        a0x = -mi.x * (b0.x + g0.x); a0y = -mi.x * (b0.y + g0.y); a0z = -mi.x * (b0.z + g0.z);
        a1x = -mi.x * (b1.x + g1.x); a1y = -mi.x * (b1.y + g1.y); a1z = -mi.x * (b1.z + g1.z);
    }
    float vx = v4.x, vy = v4.y, vz = v4.z;
    // the velocity half-phases: every lane of the warp walks through them together (chain_C is a warp-wide loop)
    // (not unrolled, and each chain routine appears once: the kernel's code stays small enough for the
    // instruction cache -- "no instruction" was the second largest stall of the unrolled version)
#pragma unroll 1
    for (int ph = 0; ph < 2; ++ph) {
        const Phase P = A.ph[ph];
        if (P.kind == 0) continue;
        const float ax = ph == 0 ? a0x : a1x, ay = ph == 0 ? a0y : a1y, az = ph == 0 ? a0z : a1z;
        if (P.kind == 1 || !JUMPS) {
            vx += P.H * ax; vy += P.H * ay; vz += P.H * az;
        } else {
            // B J / J B: the kick apart, the chains on a piecewise constant velocity
            const float cax = P.bkick ? 0.f : ax, cay = P.bkick ? 0.f : ay, caz = P.bkick ? 0.f : az;
            if (P.bkick == 1) { vx += P.H * ax; vy += P.H * ay; vz += P.H * az; }
            // slots: J' if the phase is a closing one (J'C'), then C', then J' if it is an opening one (C'J')
#pragma unroll 1
            for (int slot = 0; slot < 3; ++slot) {
                if (slot == 1) {
                    if (P.coul) chain_C<G, LOG, MECH>(m, A, live, cc, i, atom, xi, lji, mi.y, cax, cay, caz, P.H, P.streamC, P.step, vx, vy, vz, tl, gl, gshift);
                    else if (P.use_grad) { vx += P.H * cax; vy += P.H * cay; vz += P.H * caz; }
                } else if (P.lj && live && (slot == 0) == (P.reverse != 0)) {
                    chain_J(m, A, cc, i, atom, xi, lji, mi.y, P.H, P.streamJ, P.step, vx, vy, vz, tl, lead);
                }
            }
            if (P.bkick == 2) { vx += P.H * ax; vy += P.H * ay; vz += P.H * az; }
        }
    }
    if (live) {
        if (A.do_aoa && lead) {
            // positions are integrated in fp64 as hi + lo (hi = the fp32 value every pair kernel reads):
            // fp32 rounding of x (ulp(18 A) = 2e-6 A) through the stiff O-H bonds is otherwise the
            // largest noise source of the whole step
            const float4 xlo = A.xl_all[i];
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
            int ix, iy, iz;
            img_unpack(__float_as_int(xlo.w), ix, iy, iz);
            X = wrap1d(X, (double)m.box[0], (double)m.inv_box[0], ix);
            Y = wrap1d(Y, (double)m.box[1], (double)m.inv_box[1], iy);
            Z = wrap1d(Z, (double)m.box[2], (double)m.inv_box[2], iz);
            const float x = (float)X, y = (float)Y, z = (float)Z;
            A.xs_out[i] = make_float4(x, y, z, xi.w);
            A.xl_out[i] = make_float4((float)(X - (double)x), (float)(Y - (double)y), (float)(Z - (double)z),
                                      __int_as_float(img_pack(ix, iy, iz)));
            float4 xb = A.x_build[i];
            float ddx = min_image1(x, xb.x, m.box[0], m.inv_box[0]);
            float ddy = min_image1(y, xb.y, m.box[1], m.inv_box[1]);
            float ddz = min_image1(z, xb.z, m.box[2], m.inv_box[2]);
            // scaled by the atom's share of the skin (R-10c): w_i = Wc / sqrt(beta m_i); the budget is (skin/2) w_i
            const float inv_w = mi.y / m.Wc;
            disp2 = (ddx * ddx + ddy * ddy + ddz * ddz) * (inv_w * inv_w);
            bad = !(isfinite(x) && isfinite(y) && isfinite(z));
        }
        bad = bad || !(isfinite(vx) && isfinite(vy) && isfinite(vz));
        if (lead) A.vs[i] = make_float4(vx, vy, vz, v4.w);
    }
    // statistics: warp reduction -> shared-memory atomics -> one set of global atomics per CTA (thousands of warps
    // hitting the same few global counters serialise at one L2 slice)
    __shared__ unsigned s_stat[8];   // proposals, accepts, gt_attempts, expiries, max_p, max_gl, max_disp2, err
    if (threadIdx.x < 8) s_stat[threadIdx.x] = 0u;
    __syncthreads();
    unsigned err = 0;
    if (bad || tl.runaway) err |= ERR_NAN;
    if (tl.max_p > 1.f + 1e-4f || tl.max_gl > 1.f + 1e-4f) err |= ERR_BOUND;
    unsigned d2b = __reduce_max_sync(full, __float_as_uint(disp2));
    err = __reduce_or_sync(full, err);
    if (JUMPS) {
        unsigned np = __reduce_add_sync(full, tl.proposals), na = __reduce_add_sync(full, tl.accepts);
        unsigned ng = __reduce_add_sync(full, tl.gt_attempts), ne = __reduce_add_sync(full, tl.expiries);
        unsigned mp = __reduce_max_sync(full, __float_as_uint(tl.max_p));
        unsigned mg = __reduce_max_sync(full, __float_as_uint(tl.max_gl));
        if (lane == 0) {
            if (np) atomicAdd(&s_stat[0], np);
            if (na) atomicAdd(&s_stat[1], na);
            if (ng) atomicAdd(&s_stat[2], ng);
            if (ne) atomicAdd(&s_stat[3], ne);
            atomicMax(&s_stat[4], mp);
            atomicMax(&s_stat[5], mg);
        }
    }
    if (lane == 0) {
        atomicMax(&s_stat[6], d2b);
        if (err) atomicOr(&s_stat[7], err);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (JUMPS) {
            if (s_stat[0]) atomicAdd(&A.ctr->proposals, (unsigned long long)s_stat[0]);
            if (s_stat[1]) atomicAdd(&A.ctr->accepts, (unsigned long long)s_stat[1]);
            if (s_stat[2]) atomicAdd(&A.ctr->gt_attempts, (unsigned long long)s_stat[2]);
            if (s_stat[3]) atomicAdd(&A.ctr->expiries, (unsigned long long)s_stat[3]);
            if (s_stat[4] > A.ctr->max_p_bits) atomicMax(&A.ctr->max_p_bits, s_stat[4]);
            if (s_stat[5] > A.ctr->max_gl_bits) atomicMax(&A.ctr->max_gl_bits, s_stat[5]);
        }
        if (s_stat[6] > A.ctr->max_disp2_bits) atomicMax(&A.ctr->max_disp2_bits, s_stat[6]);
        // R-10c list schedule, decided here: the list kernels enqueued behind this launch run if the lists are list_P steps
        // old, or (from list_Q steps on) if some atom of this CTA is farther than its share of the skin from where they
        // saw it; such an atom with nothing to arm is an error
        const bool over = __uint_as_float(s_stat[6]) > m.half_skin2;
        const int age = A.trigger ? A.step_id - A.ctr->last_build : 0;
        if (A.trigger && (age >= A.list_P || (over && age >= A.list_Q))) A.ctr->go_step = A.step_id;
        else if (over) s_stat[7] |= ERR_SKIN;
        if (s_stat[7]) atomicOr(&A.ctr->err, s_stat[7]);
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
                       const float *__restrict__ sigma, const float *__restrict__ eps, double kT, double hs_over_wnorm,
                       float4 *__restrict__ xs, float4 *__restrict__ vs, float4 *__restrict__ xl, float2 *__restrict__ lj,
                       float2 *__restrict__ mi, float2 *__restrict__ hw, int *__restrict__ orig) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    float x = wrap1(pos[3 * i], m.box[0], m.inv_box[0]);
    float y = wrap1(pos[3 * i + 1], m.box[1], m.inv_box[1]);
    float z = wrap1(pos[3 * i + 2], m.box[2], m.inv_box[2]);
    xs[i] = make_float4(x, y, z, charge[i]);
    vs[i] = make_float4(vel[3 * i], vel[3 * i + 1], vel[3 * i + 2], 0.f);
    xl[i] = make_float4(0.f, 0.f, 0.f, __int_as_float(img_pack(0, 0, 0)));   // residual 0, image counters 0
    float e = eps[i];
    lj[i] = make_float2(e > 0.f ? (float)sqrt((double)sigma[i]) : 0.f, e > 0.f ? (float)(2.0 * sqrt((double)e)) : 0.f);
    double md = (double)mass[i];
    mi[i] = make_float2((float)(kKcal / md), (float)sqrt(md / (kT * kKcal)));
    // the atom's share of a pair's skin, (skin/2) w_i with w_i = m_i^-1/2 / mean(m^-1/2) (R-10c), as an fp64 value split in
    // two floats: list-edge ties are decided with the same number the fp64 oracle uses
    const double hsw = (1.0 / sqrt(md)) * hs_over_wnorm;
    const float hsw_hi = (float)hsw;
    hw[i] = make_float2(hsw_hi, (float)(hsw - (double)hsw_hi));
    orig[i] = i;
}

// re-read the caller's positions (wrapped) and velocities into the current sorted order
// moved (may be NULL): set to 1 when some atom is farther than skin/2 from its position at the last list build
// keep: the image counters survive (jump_refresh_lazy: the caller hands the trajectory back); an atom whose
// position is bit for bit the one the library wrote keeps its fp64 residual too, any other restarts it at 0 and adds
// the box lengths its coordinate lies outside [0, L) by.  !keep (jump_refresh): residual and counters restart at 0.
__global__ void k_reload(Model m, const float *__restrict__ pos, const float *__restrict__ vel,
                         const int *__restrict__ orig, float4 *__restrict__ xs, float4 *__restrict__ vs,
                         float4 *__restrict__ xl, const float4 *__restrict__ x_build, int *__restrict__ moved, int keep,
                         const float2 *__restrict__ mi) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int o = orig[i];
    const float4 old = xs[i];
    float4 x = old;
    const float px = pos[3 * o], py = pos[3 * o + 1], pz = pos[3 * o + 2];
    x.x = wrap1(px, m.box[0], m.inv_box[0]);
    x.y = wrap1(py, m.box[1], m.inv_box[1]);
    x.z = wrap1(pz, m.box[2], m.inv_box[2]);
    if (moved) {
        const float4 xb = x_build[i];
        const float dx = min_image1(x.x, xb.x, m.box[0], m.inv_box[0]);
        const float dy = min_image1(x.y, xb.y, m.box[1], m.inv_box[1]);
        const float dz = min_image1(x.z, xb.z, m.box[2], m.inv_box[2]);
        const float inv_w = mi[i].y / m.Wc;   // (the atom's budget is (skin/2) w_i, R-10c)
        const float d2 = (dx * dx + dy * dy + dz * dz) * (inv_w * inv_w);
        if (!(d2 <= m.half_skin2)) *moved = 1;   // also when a position is not finite
    }
    float4 l = make_float4(0.f, 0.f, 0.f, __int_as_float(img_pack(0, 0, 0)));
    if (keep) {
        const float4 lo = xl[i];
        if (x.x == old.x && x.y == old.y && x.z == old.z) l = lo;
        else {
            int ix, iy, iz;
            img_unpack(__float_as_int(lo.w), ix, iy, iz);
            ix += (int)floorf(px * m.inv_box[0]); iy += (int)floorf(py * m.inv_box[1]); iz += (int)floorf(pz * m.inv_box[2]);
            l.w = __int_as_float(img_pack(ix, iy, iz));
        }
    }
    xs[i] = x;
    xl[i] = l;
    vs[i] = make_float4(vel[3 * o], vel[3 * o + 1], vel[3 * o + 2], 0.f);
}

// image counters (sorted) -> caller order, n x 3 int32
__global__ void k_images(int n, const float4 *__restrict__ xl, const int *__restrict__ orig, int *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int ix, iy, iz;
    img_unpack(__float_as_int(xl[i].w), ix, iy, iz);
    int o = orig[i];
    out[3 * o] = ix; out[3 * o + 1] = iy; out[3 * o + 2] = iz;
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
static void update_dispatch(const Model &m, const UpdateArgs &A, cudaStream_t st) {
    const int B = 128;
    const unsigned grid = (unsigned)(((long long)m.n * G + B - 1) / B);
    if (m.eps_adaptive) {
        if (A.events) k_update<true, G, true, 1><<<grid, B, 0, st>>>(m, A);
        else k_update<true, G, false, 1><<<grid, B, 0, st>>>(m, A);
    } else if (m.combined) {
        if (A.events) k_update<true, G, true, 2><<<grid, B, 0, st>>>(m, A);
        else k_update<true, G, false, 2><<<grid, B, 0, st>>>(m, A);
    } else {
        if (A.events) k_update<true, G, true, 0><<<grid, B, 0, st>>>(m, A);
        else k_update<true, G, false, 0><<<grid, B, 0, st>>>(m, A);
    }
}
// lanes per jump chain: as many as keep the whole grid resident at once (SMs x resident CTAs of k_update x 128
// threads, asked of the occupancy API); A.lanes != 0 (jump_set_lanes: 1, 4, 8, 16) overrides, for tests and experiments
static int lanes_per_chain(int n, int forced) {
    if (forced == 1 || forced == 4 || forced == 8 || forced == 16) return forced;
    static long long budget = 0;
    if (budget == 0) {
        int dev = 0, sms = 148, per_sm = 6;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_update<true, 8, false, 0>, 128, 0) != cudaSuccess || per_sm < 1)
            per_sm = 6;
        budget = (long long)sms * per_sm * 128;
    }
    if ((long long)n * 16 <= budget) return 16;
    if ((long long)n * 8 <= budget) return 8;
    if ((long long)n * 4 <= budget) return 4;
    return 1;
}
void launch_update(const Model &m, const UpdateArgs &A, bool jumps, cudaStream_t st, int64_t *launches) {
    if (!jumps) {
        const int B = 128;
        k_update<false, 1, false, 0><<<(unsigned)((m.n + B - 1) / B), B, 0, st>>>(m, A);
    } else {
        switch (lanes_per_chain(m.n, A.lanes)) {
            case 16: update_dispatch<16>(m, A, st); break;
            case 8: update_dispatch<8>(m, A, st); break;
            case 4: update_dispatch<4>(m, A, st); break;
            default: update_dispatch<1>(m, A, st); break;
        }
    }
    *launches += 1;
}
void launch_writeback(int n, const float4 *xs, const float4 *vs, const int *orig, float *pos, float *vel, cudaStream_t st,
                      int64_t *launches) {
    k_writeback<<<(n + 255) / 256, 256, 0, st>>>(n, xs, vs, orig, pos, vel);
    *launches += 1;
}
void launch_load(const Model &m, const float *pos, const float *vel, const float *mass, const float *charge,
                 const float *sigma, const float *eps, double kT, double hs_over_wnorm, float4 *xs, float4 *vs, float4 *xl, float2 *lj,
                 float2 *mi, float2 *hw, int *orig, cudaStream_t st, int64_t *launches) {
    k_load<<<(m.n + 255) / 256, 256, 0, st>>>(m, pos, vel, mass, charge, sigma, eps, kT, hs_over_wnorm, xs, vs, xl, lj, mi, hw, orig);
    *launches += 1;
}
void launch_reload(const Model &m, const float *pos, const float *vel, const int *orig, float4 *xs, float4 *vs,
                   float4 *xl, const float4 *x_build, int *moved, int keep, const float2 *mi, cudaStream_t st, int64_t *launches) {
    k_reload<<<(m.n + 255) / 256, 256, 0, st>>>(m, pos, vel, orig, xs, vs, xl, x_build, moved, keep, mi);
    *launches += 1;
}
void launch_images(int n, const float4 *xl, const int *orig, int *out, cudaStream_t st, int64_t *launches) {
    k_images<<<(n + 255) / 256, 256, 0, st>>>(n, xl, orig, out);
    *launches += 1;
}
void launch_kinetic(int n, const float4 *vs, const float2 *mi, double *out, cudaStream_t st, int64_t *launches) {
    k_kinetic<<<(n + 255) / 256, 256, 0, st>>>(n, vs, mi, out);
    *launches += 1;
}

}  // namespace jb
