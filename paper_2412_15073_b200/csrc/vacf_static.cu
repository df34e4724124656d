// vacf_static.cu -- jump_vacf_dot_static: the velocity autocorrelation sum of observe.cu (k_vacf_dot + k_vacf_final,
// P:L529-531, L583-589) for callers that may not allocate: code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  The per-CTA partial sums live in a file-scope __device__ array instead of a
// buffer of the context, so the entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// The array (256 KiB) is part of the library's device image: every GPU that loads the library holds it until the
// process exits.  In HOST code its name is a host-side stand-in, not a device address -- the address a kernel may be
// given comes from cudaGetSymbolAddress, taken once per device with that device current (static_setup below).
// Every call on a device shares the array: two calls that overlap on the GPU (different streams, no dependency
// between them) race on it.  Nothing in it has to start at zero: a call with n atoms overwrites its first
// ceil(n / 256) partial sums before its second kernel reads exactly those.
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include <string>
#include "../../include/jump_b200.h"

namespace {

constexpr int kThreads = 256;
constexpr int kMaxParts = JUMP_VACF_STATIC_MAX_ATOMS / kThreads;   // 16384 partial sums of 16 B: 256 KiB
static_assert(JUMP_VACF_STATIC_MAX_ATOMS % kThreads == 0, "the limit is a whole number of CTAs");

static __device__ __align__(256) double2 g_vacf_part[kMaxParts];

constexpr int kMaxDevices = 64;
std::mutex g_lock;
double2 *g_part_addr[kMaxDevices];   // device address of g_vacf_part on each device, 0 until static_setup ran there
thread_local std::string t_err;

// per-CTA partial sums in fp64, in a fixed order (shared-memory tree): (sum of dots, number of selected atoms).
// v_now / v_origin: n x 3 packed floats in the same atom order; select: 0 / non-zero per atom, or null (all atoms).
__global__ void __launch_bounds__(kThreads) k_vacf_dot_static(int n, const float *__restrict__ v_now,
                                                              const float *__restrict__ v_origin,
                                                              const int32_t *__restrict__ select, double2 *__restrict__ part) {
    __shared__ double s_d[kThreads], s_c[kThreads];
    const int i = blockIdx.x * kThreads + threadIdx.x;
    double d = 0.0, cnt = 0.0;
    if (i < n && (!select || select[i] != 0)) {
        const float *a = v_origin + 3 * (size_t)i, *b = v_now + 3 * (size_t)i;
        d = (double)a[0] * (double)b[0] + (double)a[1] * (double)b[1] + (double)a[2] * (double)b[2];
        cnt = 1.0;
    }
    s_d[threadIdx.x] = d; s_c[threadIdx.x] = cnt;
    __syncthreads();
    for (int off = kThreads / 2; off > 0; off >>= 1) {
        if (threadIdx.x < off) { s_d[threadIdx.x] += s_d[threadIdx.x + off]; s_c[threadIdx.x] += s_c[threadIdx.x + off]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = make_double2(s_d[0], s_c[0]);
}

// out[0] = sum / count (0 when nothing is selected), out[1] = count
__global__ void __launch_bounds__(kThreads) k_vacf_final_static(int nb, const double2 *__restrict__ part, double *__restrict__ out) {
    __shared__ double s_d[kThreads], s_c[kThreads];
    double d = 0.0, c = 0.0;
    for (int t = threadIdx.x; t < nb; t += kThreads) { d += part[t].x; c += part[t].y; }
    s_d[threadIdx.x] = d; s_c[threadIdx.x] = c;
    __syncthreads();
    for (int off = kThreads / 2; off > 0; off >>= 1) {
        if (threadIdx.x < off) { s_d[threadIdx.x] += s_d[threadIdx.x + off]; s_c[threadIdx.x] += s_c[threadIdx.x + off]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = s_c[0] > 0.0 ? s_d[0] / s_c[0] : 0.0; out[1] = s_c[0]; }
}

int fail(int code, const std::string &what) { t_err = what; return code; }

// once per device, with that device current: the device address of the scratch array
int static_setup(double2 **addr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(JUMP_E_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(JUMP_E_ARG, "device ordinal beyond 63");
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_part_addr[dev]) {
        double2 *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_vacf_part);
        if (e != cudaSuccess || !p) return fail(JUMP_E_CUDA, std::string("cudaGetSymbolAddress(g_vacf_part): ") + cudaGetErrorString(e));
        g_part_addr[dev] = p;
    }
    if (addr) *addr = g_part_addr[dev];
    return 0;
}

}  // namespace

extern "C" int jump_vacf_static_setup(void) { return static_setup(nullptr); }

extern "C" const char *jump_vacf_static_last_error(void) { return t_err.c_str(); }

extern "C" int jump_vacf_dot_static(int32_t n, const float *d_v_now, const float *d_v_origin, const int32_t *d_select,
                                    double *d_out, void *stream) {
    if (n <= 0 || !d_v_now || !d_v_origin || !d_out) return fail(JUMP_E_ARG, "jump_vacf_dot_static: n <= 0 or a null array");
    if (n > JUMP_VACF_STATIC_MAX_ATOMS)
        return fail(JUMP_E_ARG, "jump_vacf_dot_static: n = " + std::to_string(n) + " atoms is beyond JUMP_VACF_STATIC_MAX_ATOMS = " +
                                    std::to_string(JUMP_VACF_STATIC_MAX_ATOMS) + " (the static scratch array holds one partial sum per 256 atoms)");
    double2 *part = nullptr;
    int r = static_setup(&part);
    if (r) return r;
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = (n + kThreads - 1) / kThreads;
    k_vacf_dot_static<<<nb, kThreads, 0, st>>>(n, d_v_now, d_v_origin, d_select, part);
    k_vacf_final_static<<<1, kThreads, 0, st>>>(nb, part, d_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(JUMP_E_CUDA, std::string("jump_vacf_dot_static launch: ") + cudaGetErrorString(e));
    return 0;
}
