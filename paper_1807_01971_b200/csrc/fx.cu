// fx.cu -- context, the vector primitives, the exact-dot kernel, the dG apply kernel and their C ABI (include/fx.h).
// sm_100a only.  Compile with -fmad=false: every FMA below is written explicitly.

#include <cstdlib>
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include "fx_internal.h"

// ------------------------------------------------------------------------------------------------------------
// context and errors
// ------------------------------------------------------------------------------------------------------------

static thread_local char g_err[512] = "";
static FxCtx g_ctx = {};

void fx_set_error(const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
}
fx_status fx_cuda_fail(cudaError_t e, const char* what) {
    fx_set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return FX_ECUDA;
}
extern "C" const char* fx_last_error(void) { return g_err; }

FxCtx* fx_ctx() {
    FxCtx* c = &g_ctx;
    if (c->ready) return c;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        fx_set_error("no CUDA device: %s (libfx has no CPU fallback)", cudaGetErrorString(e));
        return nullptr;
    }
    if (cudaGetDevice(&c->device) != cudaSuccess) { fx_set_error("cudaGetDevice failed"); return nullptr; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) { fx_set_error("cudaGetDeviceProperties failed"); return nullptr; }
    c->num_sms = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : FX_NUM_SMS_DEFAULT;
    const size_t ex_bytes = (FX_NDIG + FX_NLIMB) * sizeof(fx_u64) + 64;
    char* base = nullptr;
    if (cudaMalloc(&base, ex_bytes) != cudaSuccess || cudaMemset(base, 0, ex_bytes) != cudaSuccess ||
        cudaMalloc(&c->result_dev, 8 * sizeof(double)) != cudaSuccess ||
        cudaMallocHost(&c->result_pinned, 8 * sizeof(double)) != cudaSuccess) {
        fx_set_error("device scratch allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    c->ex.dig = (fx_u64*)base;
    c->ex.limbs = c->ex.dig + FX_NDIG;
    c->ex.flags = (int*)(c->ex.limbs + FX_NLIMB);
    c->ex.ticket = (unsigned int*)(c->ex.flags + 4);
    c->cg_fused = 1;
    { const char* e = getenv("FX_PDL"); c->cg_pdl = e && e[0] == '1'; }      // measured slower on B200: off unless asked for
    c->ready = true;
    return c;
}

extern "C" fx_status fx_set_stream(void* s) {
    FxCtx* c = fx_ctx();
    if (!c) return FX_ECUDA;
    c->stream = (cudaStream_t)s;
    return FX_OK;
}

extern "C" fx_status fx_set_launch(int32_t id, int32_t grid_dim, int32_t block_dim) {
    if (id < 0 || id > 3 || grid_dim < 0 || block_dim < 0 || block_dim > 1024 || (block_dim & 31)) {
        fx_set_error("fx_set_launch: bad arguments"); return FX_EINVAL;
    }
    g_ctx.launch[id][0] = grid_dim; g_ctx.launch[id][1] = block_dim;
    return FX_OK;
}
extern "C" fx_status fx_set_cg_fused(int32_t fused) {
    if (fused < 0 || fused > 3) { fx_set_error("fx_set_cg_fused: mode must be 0..3"); return FX_EINVAL; }
    if (!g_ctx.ready && !fx_ctx()) return FX_ECUDA;
    g_ctx.cg_fused = fused;
    return FX_OK;
}
extern "C" fx_status fx_set_dg_path(int32_t path) {
    if (path < 0 || path > 2) { fx_set_error("fx_set_dg_path: path must be 0..2"); return FX_EINVAL; }
    if (!g_ctx.ready && !fx_ctx()) return FX_ECUDA;
    g_ctx.dg_path = path;
    return FX_OK;
}
extern "C" int64_t fx_launch_count(void) { return g_ctx.launches; }

extern "C" void fx_shutdown(void) {
    FxCtx* c = &g_ctx;
    if (!c->ready) return;
    cudaStreamSynchronize(c->stream);
    cudaFree(c->ex.dig); cudaFree(c->result_dev); cudaFreeHost(c->result_pinned);
    if (c->cg_vec) cudaFree(c->cg_vec);
    if (c->cg_scal) cudaFree(c->cg_scal);
    if (c->cg_pdig) cudaFree(c->cg_pdig);
    if (c->ara_vec) cudaFree(c->ara_vec);
    if (c->cg_scal_pinned) cudaFreeHost(c->cg_scal_pinned);
    for (int i = 0; i < 4; ++i) if (c->stage[i]) cudaFree(c->stage[i]);
    if (c->copy_stream) { cudaStreamDestroy(c->copy_stream); for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_copy[i]); cudaEventDestroy(c->ev_comp[i]); } }
    int64_t l = c->launches;
    memset(c, 0, sizeof(*c));
    c->launches = l;
}


// ------------------------------------------------------------------------------------------------------------
// axpby, pointwise_dot  (section 3.2; canonical order DESIGN.md 3.2)
// HBM roofline: 24 B per element (16 B when beta == 0 / 32 B for pointwise with beta != 0), 1-3 fp64 ops.
// ------------------------------------------------------------------------------------------------------------

template <bool BETA0>
__device__ __forceinline__ double axpby1(double a, double x, double b, double y) {
    return BETA0 ? __dmul_rn(a, x) : __fma_rn(a, x, __dmul_rn(b, y));
}
template <bool BETA0>
__device__ __forceinline__ double pwd1(double a, double x1, double x2, double b, double y) {
    const double u = __dmul_rn(a, x1);
    return BETA0 ? __dmul_rn(u, x2) : __fma_rn(u, x2, __dmul_rn(b, y));
}

#define FX_EW_U 4     // 16-byte vectors per thread and array

template <bool BETA0, bool VEC>
__global__ void __launch_bounds__(1024) k_axpby(double a, const double* __restrict__ x, double b, double* y, long long n) {
    if (VEC) {
        const long long n2 = n >> 1;
        const double2* x2 = reinterpret_cast<const double2*>(x);
        double2* y2 = reinterpret_cast<double2*>(y);
        const long long tile = (long long)blockDim.x * FX_EW_U;
        for (long long base = (long long)blockIdx.x * tile; base < n2; base += (long long)gridDim.x * tile) {
            double2 xv[FX_EW_U], yv[FX_EW_U];
#pragma unroll
            for (int u = 0; u < FX_EW_U; ++u) {
                const long long i = base + (long long)u * blockDim.x + threadIdx.x;
                if (i < n2) { xv[u] = x2[i]; if (!BETA0) yv[u] = y2[i]; }
            }
#pragma unroll
            for (int u = 0; u < FX_EW_U; ++u) {
                const long long i = base + (long long)u * blockDim.x + threadIdx.x;
                if (i < n2) {
                    double2 o;
                    o.x = axpby1<BETA0>(a, xv[u].x, b, BETA0 ? 0.0 : yv[u].x);
                    o.y = axpby1<BETA0>(a, xv[u].y, b, BETA0 ? 0.0 : yv[u].y);
                    y2[i] = o;
                }
            }
        }
        if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) y[n - 1] = axpby1<BETA0>(a, x[n - 1], b, BETA0 ? 0.0 : y[n - 1]);
    } else {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
            y[i] = axpby1<BETA0>(a, x[i], b, BETA0 ? 0.0 : y[i]);
    }
}

template <bool BETA0, bool VEC>
__global__ void __launch_bounds__(1024) k_pointwise(double a, const double* __restrict__ x1, const double* __restrict__ x2,
                                                    double b, double* y, long long n) {
    if (VEC) {
        const long long n2 = n >> 1;
        const double2* p1 = reinterpret_cast<const double2*>(x1);
        const double2* p2 = reinterpret_cast<const double2*>(x2);
        double2* y2 = reinterpret_cast<double2*>(y);
        const long long tile = (long long)blockDim.x * FX_EW_U;
        for (long long base = (long long)blockIdx.x * tile; base < n2; base += (long long)gridDim.x * tile) {
            double2 av[FX_EW_U], bv[FX_EW_U], yv[FX_EW_U];
#pragma unroll
            for (int u = 0; u < FX_EW_U; ++u) {
                const long long i = base + (long long)u * blockDim.x + threadIdx.x;
                if (i < n2) { av[u] = p1[i]; bv[u] = p2[i]; if (!BETA0) yv[u] = y2[i]; }
            }
#pragma unroll
            for (int u = 0; u < FX_EW_U; ++u) {
                const long long i = base + (long long)u * blockDim.x + threadIdx.x;
                if (i < n2) {
                    double2 o;
                    o.x = pwd1<BETA0>(a, av[u].x, bv[u].x, b, BETA0 ? 0.0 : yv[u].x);
                    o.y = pwd1<BETA0>(a, av[u].y, bv[u].y, b, BETA0 ? 0.0 : yv[u].y);
                    y2[i] = o;
                }
            }
        }
        if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0)
            y[n - 1] = pwd1<BETA0>(a, x1[n - 1], x2[n - 1], b, BETA0 ? 0.0 : y[n - 1]);
    } else {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
            y[i] = pwd1<BETA0>(a, x1[i], x2[i], b, BETA0 ? 0.0 : y[i]);
    }
}

static void ew_shape(FxCtx* c, int64_t n, bool vec, int* grid, int* block) {
    int bd = c->launch[1][1] ? c->launch[1][1] : 256;
    long long per_block = (long long)bd * (vec ? 2 * FX_EW_U : 1);
    long long g = (n + per_block - 1) / per_block;
    if (g < 1) g = 1;
    const long long gmax = (long long)c->num_sms * 64;
    if (g > gmax) g = gmax;
    if (c->launch[1][0]) g = c->launch[1][0];
    *grid = (int)g; *block = bd;
}

extern "C" fx_status fx_axpby(double alpha, const double* x, double beta, double* y, int64_t n) {
    if (n < 0 || (n > 0 && (!x || !y))) { fx_set_error("fx_axpby: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    FxCtx* c = fx_ctx();
    if (!c) return FX_ECUDA;
    const bool vec = aligned16(x) && aligned16(y);
    int grid, block; ew_shape(c, n, vec, &grid, &block);
    if (beta == 0.0) { if (vec) k_axpby<true, true><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); else k_axpby<true, false><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); }
    else { if (vec) k_axpby<false, true><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); else k_axpby<false, false><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); }
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

extern "C" fx_status fx_pointwise_dot(double alpha, const double* x1, const double* x2, double beta, double* y, int64_t n) {
    if (n < 0 || (n > 0 && (!x1 || !x2 || !y))) { fx_set_error("fx_pointwise_dot: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    FxCtx* c = fx_ctx();
    if (!c) return FX_ECUDA;
    const bool vec = aligned16(x1) && aligned16(x2) && aligned16(y);
    int grid, block; ew_shape(c, n, vec, &grid, &block);
    if (beta == 0.0) { if (vec) k_pointwise<true, true><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); else k_pointwise<true, false><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); }
    else { if (vec) k_pointwise<false, true><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); else k_pointwise<false, false><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); }
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

// z <- alpha x1 y1 + beta x2 y2 + gamma z.  48 B per element (40 B for gamma == 0).
template <bool GAMMA0>
__global__ void __launch_bounds__(1024) k_pointwise2(double a, const double* __restrict__ x1, const double* __restrict__ y1, double b,
                                                     const double* __restrict__ x2, const double* __restrict__ y2, double c, double* z,
                                                     long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double u = __dmul_rn(a, x1[i]), v = __dmul_rn(b, x2[i]);
        const double t = GAMMA0 ? __dmul_rn(v, y2[i]) : __fma_rn(v, y2[i], __dmul_rn(c, z[i]));
        z[i] = __fma_rn(u, y1[i], t);
    }
}

extern "C" fx_status fx_pointwise_dot2(double alpha, const double* x1, const double* y1, double beta, const double* x2, const double* y2,
                                       double gamma, double* z, int64_t n) {
    if (n < 0 || (n > 0 && (!x1 || !y1 || !x2 || !y2 || !z))) { fx_set_error("fx_pointwise_dot2: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    FxCtx* c = fx_ctx();
    if (!c) return FX_ECUDA;
    int grid, block; ew_shape(c, n, false, &grid, &block);
    if (gamma == 0.0) k_pointwise2<true><<<grid, block, 0, c->stream>>>(alpha, x1, y1, beta, x2, y2, gamma, z, n);
    else k_pointwise2<false><<<grid, block, 0, c->stream>>>(alpha, x1, y1, beta, x2, y2, gamma, z, n);
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}
