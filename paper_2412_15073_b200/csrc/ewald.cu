// ewald.cu -- the reciprocal part of the Ewald sum as the slow many-body force F_{0,1} of the three-level
// JUMP-RESPA1 / BAOAB-RESPA1 schemes (NEXT-2, R-21).
//
//   U_rec  = (C / 2V) sum_{k != 0} (4 pi / k^2) exp(-k^2 / 4 alpha^2) |S(k)|^2,   S(k) = sum_j q_j exp(i k.x_j),
//   U_excl = -sum_{excluded pairs} C q_i q_j erf(alpha r_ij) / r_ij   (the reciprocal sum contains every pair, also
//            those R-9 keeps out of the direct sum: their smooth part is taken out again),
//   k = 2 pi (nx/Lx, ny/Ly, nz/Lz), |k| <= k_cut; k and -k give the same term, so a half space is summed.
//   d U_rec / d x_i = sum_half 2 A_k q_i k (Im S cos(k.x_i) - Re S sin(k.x_i)),  A_k = (C/V)(4 pi/k^2) exp(-k^2/4 alpha^2).
//
// The paper's SPME is an FFT approximation of this sum; the sum itself is evaluated here (O(N n_k): two passes of
// independent sincos terms, ALU-bound, no tensor-core shape).  The phase k.x / 2 pi = n.(x/L) is formed in 32-bit
// FIXED POINT: the scaled coordinate x/L in [0, 1) (from the fp64 position xs + xl) becomes an unsigned integer with
// 2^32 = one cycle, and n.(x/L) mod 1 is then three wrapping integer multiply-adds -- the reduction to one period is
// free and exact, the phase error is |n| 2^-33 <= 4e-9 cycles, and the fp64 multiply-adds, rint and the five 64-bit
// conversions per term (a 16-per-clock pipe) of an fp64 phase are gone: that form of the loops ran 1.5 times slower.  The sines
// and cosines are polynomials on [-pi/4, pi/4] after an integer quadrant reduction: fp64 in the structure-factor pass
// (S(k) is the small remainder of N cancelling charges), fp32 in the force pass.
// No floating-point atomics: structure-factor partials per atom chunk are written out and added in a fixed order, the
// force of an atom is one warp's shuffle reduction -- bitwise deterministic.
#include "launch.h"

namespace jb {

constexpr int EW_BIAS = 512;   // |n| <= 511 per dimension
__host__ __device__ inline int ew_pack(int nx, int ny, int nz) {
    return (nx + EW_BIAS) | ((ny + EW_BIAS) << 10) | ((nz + EW_BIAS) << 20);
}
__device__ inline void ew_unpack(int w, int &nx, int &ny, int &nz) {
    nx = (w & 1023) - EW_BIAS; ny = ((w >> 10) & 1023) - EW_BIAS; nz = ((w >> 20) & 1023) - EW_BIAS;
}
// scaled coordinate in [0, 1) -> 32-bit fixed point (wraps: 1.0 -> 0)
__device__ inline unsigned fix_cycle(double s) { return (unsigned)(__double2ull_rn(s * 4294967296.0) & 0xffffffffull); }
// cos and sin of 2 pi p / 2^32 for an integer phase p, with the whole range reduction in integers: q = nearest
// quarter cycle, r = p - q 2^30 in [-2^29, 2^29) i.e. theta = 2 pi r / 2^32 in [-pi/4, pi/4); least-squares
// polynomials in theta^2 made for this file (sin to 1e-8, cos to 2e-10 in exact arithmetic); the int -> fp32
// conversion rounds r to 24 bits, at most 4.7e-8 rad.  fp32: the force pass.  (sincospif cost 35 instructions, this
// costs 22: that pass is bound by instruction issue.)
__device__ inline void phase_sincos(unsigned p, float &s, float &c) {
    const unsigned q = (p + 0x20000000u) >> 30;
    const int r = (int)(p - (q << 30));
    const float th = 1.4629180792671596e-9f * (float)r;   // 2 pi / 2^32
    const float t = th * th;
    float sp = fmaf(t, -1.958794891834259e-4f, 8.332748897373676e-3f);
    sp = fmaf(t, sp, -0.166666641831398f);
    const float sn = fmaf(th * t, sp, th);
    float cp = fmaf(t, 2.4463912268402055e-5f, -1.388759003020823e-3f);
    cp = fmaf(t, cp, 4.166664928197861e-2f);
    cp = fmaf(t, cp, -0.5f);
    const float cs = fmaf(t, cp, 1.f);
    // angle = q pi/2 + theta
    const float a = (q & 1u) ? cs : sn, b = (q & 1u) ? sn : cs;
    s = (q & 2u) ? -a : a;
    c = ((q + 1u) & 2u) ? -b : b;
}
// The same in fp64 (Taylor polynomials to theta^11 / theta^12: 7e-12 on [-pi/4, pi/4]; r converts exactly), for the
// structure-factor pass: in a liquid of neutral molecules S(k) at small k is what is left of N cancelling charges
// (|S| ~ 1e-2 sqrt(N) |q| where A_k is largest), so the 6e-8 rounding of an fp32 cosine per atom came back as 3e-6 in
// S(k) and 7e-6 in every force -- the sines and cosines of this pass need more than fp32 holds.
__device__ inline void phase_sincos_d(unsigned p, double &s, double &c) {
    const unsigned q = (p + 0x20000000u) >> 30;
    const int r = (int)(p - (q << 30));
    const double th = 1.4629180792671596e-9 * (double)r;   // 2 pi / 2^32
    const double t = th * th;
    double sp = fma(t, -2.505210838544172e-8, 2.755731922398589e-6);   // -1/11!, 1/9!
    sp = fma(t, sp, -1.984126984126984e-4);                            // -1/7!
    sp = fma(t, sp, 8.333333333333333e-3);                             //  1/5!
    sp = fma(t, sp, -1.666666666666667e-1);                            // -1/3!
    const double sn = fma(th * t, sp, th);
    double cp = fma(t, 2.087675698786810e-9, -2.755731922398589e-7);   //  1/12!, -1/10!
    cp = fma(t, cp, 2.480158730158730e-5);                             //  1/8!
    cp = fma(t, cp, -1.388888888888889e-3);                            // -1/6!
    cp = fma(t, cp, 4.166666666666667e-2);                             //  1/4!
    cp = fma(t, cp, -0.5);
    const double cs = fma(t, cp, 1.0);
    const double a = (q & 1u) ? cs : sn, b = (q & 1u) ? sn : cs;
    s = (q & 2u) ? -a : a;
    c = ((q + 1u) & 2u) ? -b : b;
}

// running sum with a compensation term (Kahan)
__device__ inline void ksum(float x, float &sum, float &comp) {
    const float y = x - comp, t = sum + y;
    comp = (t - sum) - y;
    sum = t;
}

constexpr int SF_THREADS = 128;   // k-vectors per CTA of the structure-factor pass
constexpr int SF_TILE = 128;      // atoms staged per pass

// S(k) partial sums: thread = one k-vector, blockIdx.y = one chunk of atoms (staged through shared memory as scaled
// fp64 coordinates and the charge; every thread reads the same entry: broadcast).
__global__ void __launch_bounds__(SF_THREADS) k_sfac_partial(int n, int nk, int chunk, double ibx, double iby, double ibz,
                                                           const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                           const int *__restrict__ kpack, double2 *__restrict__ part) {
    __shared__ uint4 tile[SF_TILE];   // (fixed-point x/Lx, y/Ly, z/Lz, -)
    __shared__ double tile_q[SF_TILE];
    const int k = blockIdx.x * SF_THREADS + threadIdx.x;
    int nx = 0, ny = 0, nz = 0;
    if (k < nk) ew_unpack(kpack[k], nx, ny, nz);
    const int a0 = blockIdx.y * chunk, a1 = min(a0 + chunk, n);
    double sr = 0.0, si = 0.0;
    for (int b = a0; b < a1; b += SF_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < SF_TILE; t += SF_THREADS) {
            const int j = b + t;
            uint4 e = make_uint4(0u, 0u, 0u, 0u);
            double q = 0.0;   // charge 0: no contribution
            if (j < a1) {
                const float4 h = xs[j], l = xl[j];
                e = make_uint4(fix_cycle(((double)h.x + (double)l.x) * ibx), fix_cycle(((double)h.y + (double)l.y) * iby),
                               fix_cycle(((double)h.z + (double)l.z) * ibz), 0u);
                q = (double)h.w;
            }
            tile[t] = e; tile_q[t] = q;
        }
        __syncthreads();
#pragma unroll 4
        for (int t = 0; t < SF_TILE; ++t) {
            const uint4 e = tile[t];
            double s, c;
            phase_sincos_d((unsigned)nx * e.x + (unsigned)ny * e.y + (unsigned)nz * e.z, s, c);
            const double q = tile_q[t];
            sr = fma(q, c, sr);
            si = fma(q, s, si);
        }
    }
    if (k < nk) part[(size_t)blockIdx.y * nk + k] = make_double2(sr, si);
}

// S(k) = sum of the partials in chunk order; W(k) = 2 A_k S(k) for the force pass, e(k) = A_k |S(k)|^2 for the energy
__global__ void k_sfac_reduce(int nk, int nch, const double2 *__restrict__ part, const double *__restrict__ coefA,
                              double2 *__restrict__ W, double *__restrict__ ek) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nk) return;
    double sr = 0.0, si = 0.0;
    for (int c = 0; c < nch; ++c) { const double2 p = part[(size_t)c * nk + k]; sr += p.x; si += p.y; }
    const double A = coefA[k];
    W[k] = make_double2(2.0 * A * sr, 2.0 * A * si);
    ek[k] = A * (sr * sr + si * si);
}

constexpr int RF_THREADS = 256;                 // 8 warps = 8 atoms per CTA
constexpr int RF_TILE = 1024;                   // k-vectors staged per pass

// gradient of U_rec + U_excl: one warp per atom, lanes stride over the k-vectors of a staged tile, shuffle reduction
__global__ void __launch_bounds__(RF_THREADS) k_rec_force(Model m, int nk, double ibx, double iby, double ibz, double alpha,
                                                         const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                         const int *__restrict__ kpack, const double2 *__restrict__ W,
                                                         const int *__restrict__ orig, const int *__restrict__ sorted_of,
                                                         const int *__restrict__ excl_ptr, const int *__restrict__ excl_idx,
                                                         float4 *__restrict__ out) {
    // a staged k-vector: (nx, ny, nz, bits of W.x) as integers for the phase and (nx, ny, nz, W.y) as floats for the
    // products -- no conversion in the loop.  fp32 sines, products and compensated fp32 sums are enough HERE (1e-7 of
    // the force, measured): unlike S(k), an atom's sum over k is not the small remainder of a cancellation.
    __shared__ int4 s_k[RF_TILE];
    __shared__ float4 s_f[RF_TILE];
    const unsigned full = 0xffffffffu;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * (RF_THREADS / 32) + warp;
    const bool live = i < m.n;
    double X = 0.0, Y = 0.0, Z = 0.0, q = 0.0;
    if (live) {
        const float4 h = xs[i], l = xl[i];
        X = (double)h.x + (double)l.x; Y = (double)h.y + (double)l.y; Z = (double)h.z + (double)l.z; q = (double)h.w;
    }
    const unsigned ux = fix_cycle(X * ibx), uy = fix_cycle(Y * iby), uz = fix_cycle(Z * ibz);
    float fx = 0.f, fy = 0.f, fz = 0.f, cx = 0.f, cy = 0.f, cz = 0.f;   // sum of term * n per dimension, compensated
    double ew = 0.0;                        // this atom's half of its exclusion-correction energies
    for (int b = 0; b < nk; b += RF_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < RF_TILE; t += RF_THREADS) {
            int nx = 0, ny = 0, nz = 0;
            double2 w = make_double2(0.0, 0.0);
            if (b + t < nk) { ew_unpack(kpack[b + t], nx, ny, nz); w = W[b + t]; }
            s_k[t] = make_int4(nx, ny, nz, __float_as_int((float)w.x));
            s_f[t] = make_float4((float)nx, (float)ny, (float)nz, (float)w.y);
        }
        __syncthreads();
        if (!live) continue;
        const int lim = min(RF_TILE, nk - b);
#pragma unroll 2
        for (int t = lane; t < lim; t += 32) {
            const int4 kn = s_k[t];
            const float4 kf = s_f[t];
            float s, c;
            phase_sincos((unsigned)kn.x * ux + (unsigned)kn.y * uy + (unsigned)kn.z * uz, s, c);
            const float term = fmaf(kf.w, c, -__int_as_float(kn.w) * s);   // 2 A_k (Im S cos - Re S sin)
            ksum(term * kf.x, fx, cx); ksum(term * kf.y, fy, cy); ksum(term * kf.z, fz, cz);
        }
    }
    double gx = (double)fx - (double)cx, gy = (double)fy - (double)cy, gz = (double)fz - (double)cz;
    const double two_pi = 6.283185307179586476925;
    gx *= q * two_pi * ibx; gy *= q * two_pi * iby; gz *= q * two_pi * ibz;   // k = 2 pi n / L
    // exclusion correction: lane l takes the l-th, l+32-th ... excluded partner of the atom
    if (live && excl_ptr) {
        const int o = orig[i], lo = excl_ptr[o], n_ex = excl_ptr[o + 1] - lo;
        for (int e = lane; e < n_ex; e += 32) {
            const int j = sorted_of[excl_idx[lo + e]];
            const float4 h = xs[j], l = xl[j];
            double d[3] = {X - ((double)h.x + (double)l.x), Y - ((double)h.y + (double)l.y), Z - ((double)h.z + (double)l.z)};
            double r2 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double L = (double)m.box[k];
                d[k] -= L * rint(d[k] / L);
                r2 += d[k] * d[k];
            }
            const double r = sqrt(r2), ar = alpha * r, qq = kCoulomb * q * (double)h.w;
            // d/dr [-qq erf(alpha r)/r] = -qq [(2 alpha / sqrt pi) exp(-alpha^2 r^2) / r - erf(alpha r) / r^2]
            const double du = -qq * (1.1283791670955126 * alpha * exp(-ar * ar) / r - erf(ar) / r2);
            gx += du * d[0] / r; gy += du * d[1] / r; gz += du * d[2] / r;
            ew -= 0.5 * qq * erf(ar) / r;
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        gx += __shfl_xor_sync(full, gx, off); gy += __shfl_xor_sync(full, gy, off); gz += __shfl_xor_sync(full, gz, off);
        ew += __shfl_xor_sync(full, ew, off);
    }
    if (live && lane == 0) out[i] = make_float4((float)gx, (float)gy, (float)gz, (float)ew);
}

// ---- factorised form of the structure-factor pass: exp(i k.x_j) = Ex_j[nx] Ey_j[ny] Ez_j[nz] -----------------------
// Per atom and dimension the phase factors exp(2 pi i a x_j / L), a = 0 .. n_max (negative a: the conjugate), are
// tabulated once per evaluation in fp64 (E = n_max,x + n_max,y + n_max,z + 3 entries per atom: 63 on the 49 A box
// against the 16 493 terms they replace), the charge folded into Ex, entry-major [E][n] so that a tile of atoms loads
// coalesced; a term is then two complex products (10 fp64 operations instead of 14 and the integer reduction).  It is
// bound by the three 16-byte shared-memory reads per term (12 wavefronts per warp and term).  The same form of the
// force pass (fp32 tables, one atom's table per warp) was measured slower than the direct fp32 polynomial (381 against
// 370 us) and is not kept.
__global__ void k_ew_tables(int n, int E, int ex, int ey, double ibx, double iby, double ibz,
                            const float4 *__restrict__ xs, const float4 *__restrict__ xl, double2 *__restrict__ tabD,
                            float2 *__restrict__ tabF) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (long long)n * E) return;
    const int e = (int)(g / n), i = (int)(g - (long long)e * n);   // consecutive threads: consecutive atoms of one entry
    const float4 h = xs[i], l = xl[i];
    const int dim = e < ex ? 0 : (e < ex + ey ? 1 : 2);
    const int a = e - (dim == 0 ? 0 : (dim == 1 ? ex : ex + ey));
    const double xd = dim == 0 ? ((double)h.x + (double)l.x) * ibx
                               : (dim == 1 ? ((double)h.y + (double)l.y) * iby : ((double)h.z + (double)l.z) * ibz);
    double sn, cs;
    phase_sincos_d((unsigned)a * fix_cycle(xd), sn, cs);
    if (tabF) tabF[(size_t)i * E + e] = make_float2((float)cs, (float)sn);   // atom-major, without the charge: the force pass
    const double q = dim == 0 ? (double)h.w : 1.0;
    tabD[(size_t)e * n + i] = make_double2(q * cs, q * sn);
}

constexpr int SF2_THREADS = 512;   // k-vectors per CTA (the tables of an atom tile are staged once per CTA)
constexpr int SF2_TA = 16;         // atoms per staged tile: E x 16 double2 <= 48 KB for E <= 192
constexpr int SF2_EMAX = 192;

__global__ void __launch_bounds__(SF2_THREADS) k_sfac_partial_tab(int n, int nk, int chunk, int E, int ex, int ey,
                                                                const double2 *__restrict__ tabD,
                                                                const int *__restrict__ kpack, double2 *__restrict__ part) {
    extern __shared__ double2 s_tab[];   // [SF2_TA][E]: the threads of a warp differ in nz mostly -- consecutive entries
    const int k = blockIdx.x * SF2_THREADS + threadIdx.x;
    int nx = 0, ny = 0, nz = 0;
    if (k < nk) ew_unpack(kpack[k], nx, ny, nz);
    const int ox = nx, oy = ex + abs(ny), oz = ex + ey + abs(nz);
    const double sy = ny < 0 ? -1.0 : 1.0, sz = nz < 0 ? -1.0 : 1.0;   // negative n: the conjugate entry
    const int a0 = blockIdx.y * chunk, a1 = min(a0 + chunk, n);
    double sr = 0.0, si = 0.0;
    for (int b = a0; b < a1; b += SF2_TA) {
        __syncthreads();
        for (int t = threadIdx.x; t < E * SF2_TA; t += SF2_THREADS) {
            const int e = t / SF2_TA, j = b + (t - e * SF2_TA);
            s_tab[(t - e * SF2_TA) * E + e] = j < a1 ? tabD[(size_t)e * n + j] : make_double2(0.0, 0.0);   // (q = 0 in Ex: no contribution)
        }
        __syncthreads();
#pragma unroll 4
        for (int t = 0; t < SF2_TA; ++t) {
            const double2 a = s_tab[t * E + ox], bb = s_tab[t * E + oy], c = s_tab[t * E + oz];
            const double by = sy * bb.y, cy = sz * c.y;
            const double pr = fma(a.x, bb.x, -a.y * by), pi = fma(a.x, by, a.y * bb.x);
            sr = fma(pr, c.x, fma(-pi, cy, sr));
            si = fma(pr, cy, fma(pi, c.x, si));
        }
    }
    if (k < nk) part[(size_t)blockIdx.y * nk + k] = make_double2(sr, si);
}

// Register-blocked form of the factorised pass: a thread owns a 4 x 4 tile of the (ny, nz) plane at one nx -- 16 complex
// accumulators -- so that per atom 9 table reads (Ex, 4 Ey, 4 Ez) feed 88 fp64 operations instead of 3 reads per 10:
// the one-term-per-thread form above is bound by its shared-memory reads.  The host lists the tiles that hold at
// least one k-vector of the sphere (tiles[]) and maps every cube position to its place in the k list (cube2k, -1
// outside the sphere); entries of a tile outside the sphere are computed and dropped.
constexpr int SB_THREADS = 128;
constexpr int SB_TA = 16;

__global__ void __launch_bounds__(SB_THREADS) k_sfac_partial_blk(int n, int nk, int chunk, int E, int ex, int ey, int ntile,
                                                               int nmy, int nmz, const double2 *__restrict__ tabD,
                                                               const int *__restrict__ tiles, const int *__restrict__ cube2k,
                                                               double2 *__restrict__ part) {
    extern __shared__ double2 s_tab[];   // [SB_TA][E]
    const int tl = blockIdx.x * SB_THREADS + threadIdx.x;
    int nx = 0, ny0 = 0, nz0 = 0;
    if (tl < ntile) ew_unpack(tiles[tl], nx, ny0, nz0);
    int oy[4], oz[4];
    double sy[4], sz[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int ny = min(ny0 + u, nmy), nz = min(nz0 + u, nmz);   // (clamped entries are dropped at the end)
        oy[u] = ex + abs(ny); sy[u] = ny < 0 ? -1.0 : 1.0;
        oz[u] = ex + ey + abs(nz); sz[u] = nz < 0 ? -1.0 : 1.0;
    }
    double ar[4][4], ai[4][4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int w = 0; w < 4; ++w) { ar[u][w] = 0.0; ai[u][w] = 0.0; }
    const int a0 = blockIdx.y * chunk, a1 = min(a0 + chunk, n);
    for (int b = a0; b < a1; b += SB_TA) {
        __syncthreads();
        for (int t = threadIdx.x; t < E * SB_TA; t += SB_THREADS) {
            const int e = t / SB_TA, j = b + (t - e * SB_TA);
            s_tab[(t - e * SB_TA) * E + e] = j < a1 ? tabD[(size_t)e * n + j] : make_double2(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll 1
        for (int t = 0; t < SB_TA; ++t) {
            const double2 *row = s_tab + t * E;
            const double2 a = row[nx];
            double pr[4], pi[4], cr[4], ci[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const double2 bb = row[oy[u]];
                const double by = sy[u] * bb.y;
                pr[u] = fma(a.x, bb.x, -a.y * by); pi[u] = fma(a.x, by, a.y * bb.x);
                const double2 c = row[oz[u]];
                cr[u] = c.x; ci[u] = sz[u] * c.y;
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    ar[u][w] = fma(pr[u], cr[w], fma(-pi[u], ci[w], ar[u][w]));
                    ai[u][w] = fma(pr[u], ci[w], fma(pi[u], cr[w], ai[u][w]));
                }
        }
    }
    if (tl < ntile) {
        const int Y = 2 * nmy + 1, Z = 2 * nmz + 1;
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const int ny = ny0 + u, nz = nz0 + w;
                if (ny > nmy || nz > nmz) continue;
                const int k = cube2k[((size_t)nx * Y + (ny + nmy)) * Z + (nz + nmz)];
                if (k >= 0) part[(size_t)blockIdx.y * nk + k] = make_double2(ar[u][w], ai[u][w]);
            }
    }
}

// Register-blocked force pass over the same 4 x 4 tiles: W = 2 A_k S(k) is laid out per tile (entry-major [16][ntile],
// 0 outside the sphere) by k_w_tiles; one warp per atom, its fp32 phase-factor table in shared memory, lanes stride
// over the tiles: 9 table reads and 16 W reads feed 16 terms (the one-term-per-lane polynomial form: 52 instructions
// per term).  Sums: fp32 inside a tile (4 terms per accumulator), fp64 across tiles.
constexpr int FB_TT = 256;     // tiles staged per pass
constexpr int FB_EMAX = 192;

__global__ void k_w_tiles(int ntile, int nmy, int nmz, const int *__restrict__ tiles, const int *__restrict__ cube2k,
                          const double2 *__restrict__ W, float2 *__restrict__ Wt) {
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= 16 * ntile) return;
    const int e = g / ntile, tl = g - e * ntile, u = e >> 2, w = e & 3;
    int nx, ny0, nz0;
    ew_unpack(tiles[tl], nx, ny0, nz0);
    const int ny = ny0 + u, nz = nz0 + w;
    float2 v = make_float2(0.f, 0.f);
    if (ny <= nmy && nz <= nmz) {
        const int Y = 2 * nmy + 1, Z = 2 * nmz + 1;
        const int k = cube2k[((size_t)nx * Y + (ny + nmy)) * Z + (nz + nmz)];
        if (k >= 0) { const double2 ww = W[k]; v = make_float2((float)ww.x, (float)ww.y); }
    }
    Wt[g] = v;
}

__global__ void __launch_bounds__(RF_THREADS) k_rec_force_blk(Model m, int ntile, int E, int ex, int ey, int nmy, int nmz,
                                                             double ibx, double iby, double ibz, double alpha,
                                                             const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                             const float2 *__restrict__ tabF, const int *__restrict__ tiles,
                                                             const float2 *__restrict__ Wt, const int *__restrict__ orig,
                                                             const int *__restrict__ sorted_of, const int *__restrict__ excl_ptr,
                                                             const int *__restrict__ excl_idx, float4 *__restrict__ out) {
    __shared__ int s_tile[FB_TT];
    __shared__ float2 s_w[16][FB_TT];
    __shared__ float2 s_t[RF_THREADS / 32][FB_EMAX];
    const unsigned full = 0xffffffffu;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * (RF_THREADS / 32) + warp;
    const bool live = i < m.n;
    double X = 0.0, Y = 0.0, Z = 0.0, q = 0.0;
    if (live) {
        const float4 h = xs[i], l = xl[i];
        X = (double)h.x + (double)l.x; Y = (double)h.y + (double)l.y; Z = (double)h.z + (double)l.z; q = (double)h.w;
        for (int e = lane; e < E; e += 32) s_t[warp][e] = tabF[(size_t)i * E + e];
    }
    const float2 *tb = s_t[warp];
    double gx = 0.0, gy = 0.0, gz = 0.0;   // sum of term * n per dimension
    double ew = 0.0;                        // this atom's half of its exclusion-correction energies
    for (int b = 0; b < ntile; b += FB_TT) {
        __syncthreads();
        const int cnt = min(FB_TT, ntile - b);
        for (int t = threadIdx.x; t < FB_TT; t += RF_THREADS) s_tile[t] = t < cnt ? tiles[b + t] : ew_pack(0, 0, 0);
        for (int t = threadIdx.x; t < 16 * FB_TT; t += RF_THREADS) {
            const int e = t / FB_TT, tl = t - e * FB_TT;
            s_w[e][tl] = tl < cnt ? Wt[(size_t)e * ntile + b + tl] : make_float2(0.f, 0.f);
        }
        __syncthreads();
        if (!live) continue;
        for (int tl = lane; tl < cnt; tl += 32) {
            int nx, ny0, nz0;
            ew_unpack(s_tile[tl], nx, ny0, nz0);
            const float2 a = tb[nx];
            float pr[4], pi[4], cr[4], ci[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int ny = min(ny0 + u, nmy), nz = min(nz0 + u, nmz);   // (clamped entries carry W = 0)
                float2 bb = tb[ex + abs(ny)];
                if (ny < 0) bb.y = -bb.y;
                pr[u] = fmaf(a.x, bb.x, -a.y * bb.y); pi[u] = fmaf(a.x, bb.y, a.y * bb.x);
                const float2 c = tb[ex + ey + abs(nz)];
                cr[u] = c.x; ci[u] = nz < 0 ? -c.y : c.y;
            }
            float Tz = 0.f, Ty = 0.f, Tx = 0.f;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                float T = 0.f;
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const float2 ww = s_w[u * 4 + w][tl];
                    const float cs = fmaf(pr[u], cr[w], -pi[u] * ci[w]), sn = fmaf(pr[u], ci[w], pi[u] * cr[w]);   // cos, sin of k.x_i
                    const float term = fmaf(ww.y, cs, -ww.x * sn);   // 2 A_k (Im S cos - Re S sin)
                    T += term;
                    Tz = fmaf(term, (float)(nz0 + w), Tz);
                }
                Tx += T;
                Ty = fmaf(T, (float)(ny0 + u), Ty);
            }
            gx = fma((double)Tx, (double)nx, gx); gy += (double)Ty; gz += (double)Tz;
        }
    }
    const double two_pi = 6.283185307179586476925;
    gx *= q * two_pi * ibx; gy *= q * two_pi * iby; gz *= q * two_pi * ibz;   // k = 2 pi n / L
    if (live && excl_ptr) {
        const int o = orig[i], lo = excl_ptr[o], n_ex = excl_ptr[o + 1] - lo;
        for (int e = lane; e < n_ex; e += 32) {
            const int j = sorted_of[excl_idx[lo + e]];
            const float4 h = xs[j], l = xl[j];
            double d[3] = {X - ((double)h.x + (double)l.x), Y - ((double)h.y + (double)l.y), Z - ((double)h.z + (double)l.z)};
            double r2 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double L = (double)m.box[k];
                d[k] -= L * rint(d[k] / L);
                r2 += d[k] * d[k];
            }
            const double r = sqrt(r2), ar = alpha * r, qq = kCoulomb * q * (double)h.w;
            const double du = -qq * (1.1283791670955126 * alpha * exp(-ar * ar) / r - erf(ar) / r2);
            gx += du * d[0] / r; gy += du * d[1] / r; gz += du * d[2] / r;
            ew -= 0.5 * qq * erf(ar) / r;
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        gx += __shfl_xor_sync(full, gx, off); gy += __shfl_xor_sync(full, gy, off); gz += __shfl_xor_sync(full, gz, off);
        ew += __shfl_xor_sync(full, ew, off);
    }
    if (live && lane == 0) out[i] = make_float4((float)gx, (float)gy, (float)gz, (float)ew);
}

// sum of n doubles by one CTA in a fixed order (energy diagnostics)
__global__ void k_sum_doubles(int n, const double *__restrict__ in, double *__restrict__ out) {
    __shared__ double s[256];
    double a = 0.0;
    for (int t = threadIdx.x; t < n; t += 256) a += in[t];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if (threadIdx.x < off) s[threadIdx.x] += s[threadIdx.x + off];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = s[0];
}

void launch_rec_force(const Model &m, const EwaldArgs &e, const float4 *xs, const float4 *xl, const int *orig,
                      const int *sorted_of, const int *excl_ptr, const int *excl_idx, float4 *out, cudaStream_t st,
                      int64_t *launches) {
    const double ibx = 1.0 / (double)m.box[0], iby = 1.0 / (double)m.box[1], ibz = 1.0 / (double)m.box[2];
    const int chunk = (m.n + e.nch - 1) / e.nch;
    if (e.tabD) {   // factorised structure-factor pass (the tables fit): see k_ew_tables
        const int ex = e.nmax[0] + 1, ey = e.nmax[1] + 1, E = ex + ey + e.nmax[2] + 1;
        const long long tot = (long long)m.n * E;
        k_ew_tables<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(m.n, E, ex, ey, ibx, iby, ibz, xs, xl, e.tabD, e.tabF);
        if (e.ntile > 0) {
            dim3 g1((unsigned)((e.ntile + SB_THREADS - 1) / SB_THREADS), (unsigned)e.nch);
            k_sfac_partial_blk<<<g1, SB_THREADS, (size_t)E * SB_TA * sizeof(double2), st>>>(m.n, e.nk, chunk, E, ex, ey, e.ntile, e.nmax[1],
                                                                                          e.nmax[2], e.tabD, e.tiles, e.cube2k, e.part);
        } else {
            dim3 g1((unsigned)((e.nk + SF2_THREADS - 1) / SF2_THREADS), (unsigned)e.nch);
            k_sfac_partial_tab<<<g1, SF2_THREADS, (size_t)E * SF2_TA * sizeof(double2), st>>>(m.n, e.nk, chunk, E, ex, ey, e.tabD, e.kpack, e.part);
        }
        k_sfac_reduce<<<(e.nk + 255) / 256, 256, 0, st>>>(e.nk, e.nch, e.part, e.coefA, e.W, e.ek);
        if (e.ntile > 0 && e.tabF) {
            k_w_tiles<<<(16 * e.ntile + 255) / 256, 256, 0, st>>>(e.ntile, e.nmax[1], e.nmax[2], e.tiles, e.cube2k, e.W, e.Wt);
            k_rec_force_blk<<<(m.n + RF_THREADS / 32 - 1) / (RF_THREADS / 32), RF_THREADS, 0, st>>>(
                m, e.ntile, E, ex, ey, e.nmax[1], e.nmax[2], ibx, iby, ibz, e.alpha, xs, xl, e.tabF, e.tiles, e.Wt, orig, sorted_of,
                excl_ptr, excl_idx, out);
            *launches += 1;
        } else {
            k_rec_force<<<(m.n + RF_THREADS / 32 - 1) / (RF_THREADS / 32), RF_THREADS, 0, st>>>(m, e.nk, ibx, iby, ibz, e.alpha, xs, xl, e.kpack,
                                                                                                 e.W, orig, sorted_of, excl_ptr, excl_idx, out);
        }
        *launches += 4;
        return;
    }
    dim3 g1((unsigned)((e.nk + SF_THREADS - 1) / SF_THREADS), (unsigned)e.nch);
    k_sfac_partial<<<g1, SF_THREADS, 0, st>>>(m.n, e.nk, chunk, ibx, iby, ibz, xs, xl, e.kpack, e.part);
    k_sfac_reduce<<<(e.nk + 255) / 256, 256, 0, st>>>(e.nk, e.nch, e.part, e.coefA, e.W, e.ek);
    k_rec_force<<<(m.n + RF_THREADS / 32 - 1) / (RF_THREADS / 32), RF_THREADS, 0, st>>>(m, e.nk, ibx, iby, ibz, e.alpha, xs, xl, e.kpack,
                                                                                         e.W, orig, sorted_of, excl_ptr, excl_idx, out);
    *launches += 3;
}
int ewald_table_entries_max() { return SF2_EMAX; }
void launch_rec_energy(const EwaldArgs &e, double *out, cudaStream_t st, int64_t *launches) {
    k_sum_doubles<<<1, 256, 0, st>>>(e.nk, e.ek, out);
    *launches += 1;
}
int ewald_pack(int nx, int ny, int nz) { return ew_pack(nx, ny, nz); }

}  // namespace jb
