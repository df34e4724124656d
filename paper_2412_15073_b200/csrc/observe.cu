// observe.cu -- observables computed on the device from the sorted state: radial distribution
// histograms, velocity autocorrelation.  (Image counters for unwrapped trajectories live in update.cu / common.cuh.)
// The paper's evidence that JUMP samples mu and keeps the dynamics is of this kind: radial distribution functions and
// diffusion constants.
#include "launch.h"

namespace jb {

constexpr int RDF_MAX_BINS = 2048;

// Pair-distance histogram: one warp per selected atom i walks the cells within reach of r_max; every unordered pair
// (j > i in the sorted order) of selected atoms with minimum-image distance r < r_max adds one to bin
// floor(r n_bins / r_max).  Integer counts: shared-memory histogram per CTA, then 64-bit global atomics -- the
// result does not depend on the order of the additions.
__global__ void __launch_bounds__(256) k_rdf(Model m, SortGrid g, int reach0, int reach1, int reach2, int lj_only, float rmax2,
                                             float bins_per_A, int n_bins, const int *__restrict__ cell_start,
                                             const float4 *__restrict__ xs, const float2 *__restrict__ lj,
                                             unsigned long long *__restrict__ hist) {
    __shared__ unsigned s_hist[RDF_MAX_BINS];
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) s_hist[b] = 0u;
    __syncthreads();
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (i < m.n && (!lj_only || lj[i].y > 0.f)) {
        const float4 xi = xs[i];
        int c3[3], start[3], cnt[3];
        const int reach[3] = {reach0, reach1, reach2};
        c3[0] = min(max((int)floor((double)xi.x * g.scale[0]), 0), g.gn[0] - 1);
        c3[1] = min(max((int)floor((double)xi.y * g.scale[1]), 0), g.gn[1] - 1);
        c3[2] = min(max((int)floor((double)xi.z * g.scale[2]), 0), g.gn[2] - 1);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            if (2 * reach[k] + 1 >= g.gn[k]) { start[k] = 0; cnt[k] = g.gn[k]; }
            else { start[k] = (c3[k] - reach[k] + g.gn[k]) % g.gn[k]; cnt[k] = 2 * reach[k] + 1; }
        }
        for (int mz = 0; mz < cnt[2]; ++mz) {
            const int cz = (start[2] + mz) % g.gn[2];
            for (int my = 0; my < cnt[1]; ++my) {
                const int cy = (start[1] + my) % g.gn[1];
                for (int mx = 0; mx < cnt[0]; ++mx) {
                    const int cx = (start[0] + mx) % g.gn[0];
                    const int cell = (cz * g.gn[1] + cy) * g.gn[0] + cx;
                    const int beg = cell_start[cell], end = cell_start[cell + 1];
                    for (int j = beg + lane; j < end; j += 32) {
                        if (j <= i || (lj_only && !(lj[j].y > 0.f))) continue;
                        const float4 xj = xs[j];
                        const float dx = min_image1(xi.x, xj.x, m.box[0], m.inv_box[0]);
                        const float dy = min_image1(xi.y, xj.y, m.box[1], m.inv_box[1]);
                        const float dz = min_image1(xi.z, xj.z, m.box[2], m.inv_box[2]);
                        const float r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 < rmax2) atomicAdd(&s_hist[min((int)(sqrtf(r2) * bins_per_A), n_bins - 1)], 1u);
                    }
                }
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x)
        if (s_hist[b]) atomicAdd(&hist[b], (unsigned long long)s_hist[b]);
}

// Velocity autocorrelation (velocity spectra): the velocities at the time origin are kept by
// ORIGINAL atom index (the sort permutes atoms between two reads); C = (1/N_sel) sum v_i(origin) . v_i(now).
__global__ void k_vacf_mark(int n, const float4 *__restrict__ vs, const int *__restrict__ orig, float4 *__restrict__ v0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v0[orig[i]] = vs[i];
}
// per-CTA partial sums in fp64, in a fixed order (shared-memory tree): (sum of dots, number of selected atoms)
__global__ void __launch_bounds__(256) k_vacf_dot(int n, int lj_only, const float4 *__restrict__ vs, const float4 *__restrict__ v0,
                                                  const int *__restrict__ orig, const float2 *__restrict__ lj,
                                                  double2 *__restrict__ part) {
    __shared__ double s_d[256], s_c[256];
    const int i = blockIdx.x * 256 + threadIdx.x;
    double d = 0.0, cnt = 0.0;
    if (i < n && (!lj_only || lj[i].y > 0.f)) {
        const float4 a = v0[orig[i]], b = vs[i];
        d = (double)a.x * (double)b.x + (double)a.y * (double)b.y + (double)a.z * (double)b.z;
        cnt = 1.0;
    }
    s_d[threadIdx.x] = d; s_c[threadIdx.x] = cnt;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if (threadIdx.x < off) { s_d[threadIdx.x] += s_d[threadIdx.x + off]; s_c[threadIdx.x] += s_c[threadIdx.x + off]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = make_double2(s_d[0], s_c[0]);
}
__global__ void k_vacf_final(int nb, const double2 *__restrict__ part, double2 *__restrict__ out) {
    __shared__ double s_d[256], s_c[256];
    double d = 0.0, c = 0.0;
    for (int t = threadIdx.x; t < nb; t += 256) { d += part[t].x; c += part[t].y; }
    s_d[threadIdx.x] = d; s_c[threadIdx.x] = c;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if (threadIdx.x < off) { s_d[threadIdx.x] += s_d[threadIdx.x + off]; s_c[threadIdx.x] += s_c[threadIdx.x + off]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = make_double2(s_d[0], s_c[0]);
}
void launch_vacf_mark(int n, const float4 *vs, const int *orig, float4 *v0, cudaStream_t st, int64_t *launches) {
    k_vacf_mark<<<(n + 255) / 256, 256, 0, st>>>(n, vs, orig, v0);
    *launches += 1;
}
void launch_vacf_dot(int n, int lj_only, const float4 *vs, const float4 *v0, const int *orig, const float2 *lj, double2 *part,
                     double2 *out, cudaStream_t st, int64_t *launches) {
    const int nb = (n + 255) / 256;
    k_vacf_dot<<<nb, 256, 0, st>>>(n, lj_only, vs, v0, orig, lj, part);
    k_vacf_final<<<1, 256, 0, st>>>(nb, part, out);
    *launches += 2;
}

// Mean-square displacement on unwrapped positions (the diffusion constants of P:L527, L575-581 are its slope / 6): the
// unwrapped position x + image * box (fp64: hi + lo + image counters, see update.cu) at the time origin is kept by
// ORIGINAL atom index; MSD = (1/N_sel) sum |x_i(now) - x_i(origin)|^2, per-CTA partial sums in a fixed order.
__device__ inline void unwrapped(const Model &m, const float4 *__restrict__ xs, const float4 *__restrict__ xl, int i, double out[3]) {
    const float4 a = xs[i], b = xl[i];
    int ix, iy, iz;
    img_unpack(__float_as_int(b.w), ix, iy, iz);
    out[0] = (double)a.x + (double)b.x + (double)ix * (double)m.box[0];
    out[1] = (double)a.y + (double)b.y + (double)iy * (double)m.box[1];
    out[2] = (double)a.z + (double)b.z + (double)iz * (double)m.box[2];
}
__global__ void k_msd_mark(Model m, const float4 *__restrict__ xs, const float4 *__restrict__ xl, const int *__restrict__ orig,
                           double *__restrict__ x0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    double u[3];
    unwrapped(m, xs, xl, i, u);
    const size_t o = 3 * (size_t)orig[i];
    x0[o] = u[0]; x0[o + 1] = u[1]; x0[o + 2] = u[2];
}
__global__ void __launch_bounds__(256) k_msd_sum(Model m, int lj_only, const float4 *__restrict__ xs, const float4 *__restrict__ xl,
                                                 const int *__restrict__ orig, const float2 *__restrict__ lj,
                                                 const double *__restrict__ x0, double2 *__restrict__ part) {
    __shared__ double s_d[256], s_c[256];
    const int i = blockIdx.x * 256 + threadIdx.x;
    double d = 0.0, cnt = 0.0;
    if (i < m.n && (!lj_only || lj[i].y > 0.f)) {
        double u[3];
        unwrapped(m, xs, xl, i, u);
        const size_t o = 3 * (size_t)orig[i];
        const double dx = u[0] - x0[o], dy = u[1] - x0[o + 1], dz = u[2] - x0[o + 2];
        d = dx * dx + dy * dy + dz * dz;
        cnt = 1.0;
    }
    s_d[threadIdx.x] = d; s_c[threadIdx.x] = cnt;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
        if (threadIdx.x < off) { s_d[threadIdx.x] += s_d[threadIdx.x + off]; s_c[threadIdx.x] += s_c[threadIdx.x + off]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = make_double2(s_d[0], s_c[0]);
}
void launch_msd_mark(const Model &m, const float4 *xs, const float4 *xl, const int *orig, double *x0, cudaStream_t st, int64_t *launches) {
    k_msd_mark<<<(m.n + 255) / 256, 256, 0, st>>>(m, xs, xl, orig, x0);
    *launches += 1;
}
void launch_msd_sum(const Model &m, int lj_only, const float4 *xs, const float4 *xl, const int *orig, const float2 *lj, const double *x0,
                    double2 *part, double2 *out, cudaStream_t st, int64_t *launches) {
    const int nb = (m.n + 255) / 256;
    k_msd_sum<<<nb, 256, 0, st>>>(m, lj_only, xs, xl, orig, lj, x0, part);
    k_vacf_final<<<1, 256, 0, st>>>(nb, part, out);
    *launches += 2;
}

int launch_rdf(const Model &m, const SortGrid &g, int lj_only, double r_max, double r_reach, int n_bins, const int *cell_start,
               const float4 *xs, const float2 *lj, unsigned long long *hist, cudaStream_t st, int64_t *launches) {
    if (n_bins <= 0 || n_bins > RDF_MAX_BINS || !(r_max > 0.0)) return -1;
    int reach[3];
    for (int k = 0; k < 3; ++k) {
        if (r_max > 0.5 * (double)m.box[k]) return -1;   // minimum image
        reach[k] = (int)ceil(r_reach / ((double)m.box[k] / g.gn[k]));   // r_reach >= r_max: see jump_rdf_accumulate
    }
    const int B = 256;
    k_rdf<<<(unsigned)(((long long)m.n * 32 + B - 1) / B), B, 0, st>>>(m, g, reach[0], reach[1], reach[2], lj_only,
                                                                   (float)(r_max * r_max), (float)(n_bins / r_max), n_bins,
                                                                   cell_start, xs, lj, hist);
    *launches += 1;
    return 0;
}

}  // namespace jb
