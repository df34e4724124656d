// observe.cu -- observables computed on the device from the sorted state: radial distribution
// histograms.  (Image counters for unwrapped trajectories live in update.cu / common.cuh.)
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
