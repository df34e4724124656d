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
// independent sincos terms, ALU-bound, no tensor-core shape).  The phase k.x / 2 pi = n.(x/L) is formed in fp64 from
// x = xs + xl and reduced to [-1/2, 1/2] before the fp32 sincospi: |n.(x/L)| reaches 30 and an fp32 phase would
// carry 2e-6 cycles of error.  No floating-point atomics: structure-factor partials per atom chunk are written out
// and added in a fixed order, the force of an atom is one warp's shuffle reduction -- bitwise deterministic.
#include "launch.h"

namespace jb {

constexpr int EW_BIAS = 512;   // |n| <= 511 per dimension
__host__ __device__ inline int ew_pack(int nx, int ny, int nz) {
    return (nx + EW_BIAS) | ((ny + EW_BIAS) << 10) | ((nz + EW_BIAS) << 20);
}
__device__ inline void ew_unpack(int w, int &nx, int &ny, int &nz) {
    nx = (w & 1023) - EW_BIAS; ny = ((w >> 10) & 1023) - EW_BIAS; nz = ((w >> 20) & 1023) - EW_BIAS;
}
// cos and sin of 2 pi t for an fp64 phase t in cycles: fp32 sincospi of the reduced phase rounded to fp32, then one
// first-order step over what the rounding dropped (up to 3e-8 cycles = 2e-7 in the sine: per-atom sums of thousands
// of such terms cancel to a small force, and that error alone used the whole 1e-5 budget of R-16)
__device__ inline void phase_sincos(double t, float &s, float &c) {
    t -= rint(t);
    const float tf = (float)t;
    const float d = 6.2831853f * (float)(t - (double)tf);
    float s0, c0;
    sincospif(2.f * tf, &s0, &c0);
    s = fmaf(d, c0, s0);
    c = fmaf(-d, s0, c0);
}

constexpr int SF_THREADS = 128;   // k-vectors per CTA of the structure-factor pass
constexpr int SF_TILE = 128;      // atoms staged per pass

// S(k) partial sums: thread = one k-vector, blockIdx.y = one chunk of atoms (staged through shared memory as scaled
// fp64 coordinates and the charge; every thread reads the same entry: broadcast).
__global__ void __launch_bounds__(SF_THREADS) k_sfac_partial(int n, int nk, int chunk, double ibx, double iby, double ibz,
                                                           const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                           const int *__restrict__ kpack, double2 *__restrict__ part) {
    __shared__ double4 tile[SF_TILE];
    const int k = blockIdx.x * SF_THREADS + threadIdx.x;
    int nx = 0, ny = 0, nz = 0;
    if (k < nk) ew_unpack(kpack[k], nx, ny, nz);
    const double dnx = (double)nx, dny = (double)ny, dnz = (double)nz;
    const int a0 = blockIdx.y * chunk, a1 = min(a0 + chunk, n);
    double sr = 0.0, si = 0.0;
    for (int b = a0; b < a1; b += SF_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < SF_TILE; t += SF_THREADS) {
            const int j = b + t;
            double4 e = make_double4(0.0, 0.0, 0.0, 0.0);
            if (j < a1) {
                const float4 h = xs[j], l = xl[j];
                e = make_double4(((double)h.x + (double)l.x) * ibx, ((double)h.y + (double)l.y) * iby,
                                 ((double)h.z + (double)l.z) * ibz, (double)h.w);
            }
            tile[t] = e;
        }
        __syncthreads();
        const int lim = min(SF_TILE, a1 - b);
#pragma unroll 4
        for (int t = 0; t < lim; ++t) {
            const double4 e = tile[t];
            float s, c;
            phase_sincos(fma(dnx, e.x, fma(dny, e.y, dnz * e.z)), s, c);
            sr = fma(e.w, (double)c, sr);
            si = fma(e.w, (double)s, si);
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
    __shared__ int s_k[RF_TILE];
    __shared__ double2 s_w[RF_TILE];
    const unsigned full = 0xffffffffu;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * (RF_THREADS / 32) + warp;
    const bool live = i < m.n;
    double X = 0.0, Y = 0.0, Z = 0.0, q = 0.0;
    if (live) {
        const float4 h = xs[i], l = xl[i];
        X = (double)h.x + (double)l.x; Y = (double)h.y + (double)l.y; Z = (double)h.z + (double)l.z; q = (double)h.w;
    }
    const double sx = X * ibx, sy = Y * iby, sz = Z * ibz;
    double gx = 0.0, gy = 0.0, gz = 0.0;   // sum of term * n per dimension
    double ew = 0.0;                        // this atom's half of its exclusion-correction energies
    for (int b = 0; b < nk; b += RF_TILE) {
        __syncthreads();
        for (int t = threadIdx.x; t < RF_TILE; t += RF_THREADS) {
            const bool in = b + t < nk;
            s_k[t] = in ? kpack[b + t] : ew_pack(0, 0, 0);
            s_w[t] = in ? W[b + t] : make_double2(0.0, 0.0);
        }
        __syncthreads();
        if (!live) continue;
        const int lim = min(RF_TILE, nk - b);
#pragma unroll 2
        for (int t = lane; t < lim; t += 32) {
            int nx, ny, nz;
            ew_unpack(s_k[t], nx, ny, nz);
            const double2 w = s_w[t];
            float s, c;
            phase_sincos(fma((double)nx, sx, fma((double)ny, sy, (double)nz * sz)), s, c);
            const double term = w.y * (double)c - w.x * (double)s;   // 2 A_k (Im S cos - Re S sin)
            gx = fma(term, (double)nx, gx); gy = fma(term, (double)ny, gy); gz = fma(term, (double)nz, gz);
        }
    }
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
    dim3 g1((unsigned)((e.nk + SF_THREADS - 1) / SF_THREADS), (unsigned)e.nch);
    k_sfac_partial<<<g1, SF_THREADS, 0, st>>>(m.n, e.nk, chunk, ibx, iby, ibz, xs, xl, e.kpack, e.part);
    k_sfac_reduce<<<(e.nk + 255) / 256, 256, 0, st>>>(e.nk, e.nch, e.part, e.coefA, e.W, e.ek);
    k_rec_force<<<(m.n + RF_THREADS / 32 - 1) / (RF_THREADS / 32), RF_THREADS, 0, st>>>(m, e.nk, ibx, iby, ibz, e.alpha, xs, xl, e.kpack,
                                                                                         e.W, orig, sorted_of, excl_ptr, excl_idx, out);
    *launches += 3;
}
void launch_rec_energy(const EwaldArgs &e, double *out, cudaStream_t st, int64_t *launches) {
    k_sum_doubles<<<1, 256, 0, st>>>(e.nk, e.ek, out);
    *launches += 1;
}
int ewald_pack(int nx, int ny, int nz) { return ew_pack(nx, ny, nz); }

}  // namespace jb
