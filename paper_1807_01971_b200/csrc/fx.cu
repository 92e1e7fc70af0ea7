// fx.cu -- context, the vector primitives, the exact-dot kernel, the dG apply kernel and their C ABI (include/fx.h).
// sm_100a only.  Compile with -fmad=false: every FMA below is written explicitly.

#include <atomic>
#include <cstdlib>
#include <mutex>
#include <new>
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include "fx_internal.h"

// ------------------------------------------------------------------------------------------------------------
// context and errors
// ------------------------------------------------------------------------------------------------------------

static thread_local char g_err[512] = "";

void fx_set_error(const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
}
fx_status fx_cuda_fail(cudaError_t e, const char* what) {
    fx_set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return FX_ECUDA;
}
extern "C" const char* fx_last_error(void) { return g_err; }

// ---- contexts (the paper's user holds typed device vectors and selects the backend per vector type, P:124, P:137:
// here the context is what carries the device and the stream) -------------------------------------------------------------
#define FX_MAX_DEV 64
static std::mutex g_mu;                        // guards the default-context table only
static FxCtx* g_default[FX_MAX_DEV] = {};
static std::atomic<long long> g_launches_freed{0};   // launches of destroyed contexts (fx_launch_count is a process total)
static std::atomic<int> g_live{0};
static FxCtx* g_all[256] = {};                 // live contexts (for fx_launch_count); guarded by g_mu

static void ctx_release(FxCtx* c) {
    if (!c) return;
    if (c->ready) {
        FxDeviceGuard guard(c);
        cudaStreamSynchronize(c->stream);
        if (c->ex.dig) cudaFree(c->ex.dig);
        if (c->result_dev) cudaFree(c->result_dev);
        if (c->result_pinned) cudaFreeHost(c->result_pinned);
        if (c->cg_vec) cudaFree(c->cg_vec);
        if (c->cg_scal) cudaFree(c->cg_scal);
        if (c->cg_pdig) cudaFree(c->cg_pdig);
        if (c->ara_vec) cudaFree(c->ara_vec);
        if (c->cg_tile) free(c->cg_tile);
        if (c->cg_scal_pinned) { cudaFreeHost(c->cg_scal_pinned); cudaEventDestroy(c->cg_ev[0]); cudaEventDestroy(c->cg_ev[1]); }
        for (int i = 0; i < 4; ++i) if (c->stage[i]) cudaFree(c->stage[i]);
        if (c->copy_stream) { cudaStreamDestroy(c->copy_stream); for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_copy[i]); cudaEventDestroy(c->ev_comp[i]); } }
        if (c->prof_ev) {
            for (int i = 0; i < 4 * c->prof_cap; ++i) cudaEventDestroy(c->prof_ev[i]);
            free(c->prof_ev);
            cudaEventDestroy(c->prof_loop[0]); cudaEventDestroy(c->prof_loop[1]);
        }
    }
    g_launches_freed += c->launches;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (int i = 0; i < 256; ++i) if (g_all[i] == c) g_all[i] = nullptr;
    }
    c->ready = false;
    delete c;
}

static fx_status ctx_make(FxCtx** out, int device, void* stream) {
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        fx_set_error("no CUDA device: %s (libfx has no CPU fallback)", cudaGetErrorString(e));
        return FX_ECUDA;
    }
    if (device < 0 || device >= ndev || device >= FX_MAX_DEV) { fx_set_error("fx_create: no device %d", device); return FX_EINVAL; }
    FxCtx* c = new (std::nothrow) FxCtx();
    if (!c) { fx_set_error("out of host memory"); return FX_ENOMEM; }
    c->device = device;
    c->stream = (cudaStream_t)stream;
    FxDeviceGuard guard(c);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { fx_set_error("cudaGetDeviceProperties failed"); delete c; return FX_ECUDA; }
    c->num_sms = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : FX_NUM_SMS_DEFAULT;
    const size_t ex_bytes = (FX_NDIG + FX_NLIMB) * sizeof(fx_u64) + 64 + 4 * sizeof(fx_u64);
    char* base = nullptr;
    if (cudaMalloc(&base, ex_bytes) != cudaSuccess || cudaMemset(base, 0, ex_bytes) != cudaSuccess ||
        cudaMalloc(&c->result_dev, 8 * sizeof(double)) != cudaSuccess ||
        cudaMallocHost(&c->result_pinned, 8 * sizeof(double)) != cudaSuccess) {
        fx_set_error("device scratch allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (base) cudaFree(base);
        if (c->result_dev) cudaFree(c->result_dev);
        delete c;
        return FX_ENOMEM;
    }
    c->ex.dig = (fx_u64*)base;
    c->ex.limbs = c->ex.dig + FX_NDIG;
    c->ex.flags = (int*)(c->ex.limbs + FX_NLIMB);
    c->ex.ticket = (unsigned int*)(c->ex.flags + 4);
    c->ex.stats = (fx_u64*)(base + (FX_NDIG + FX_NLIMB) * sizeof(fx_u64) + 64);
    c->cg_fused = 1;
    { const char* ev = getenv("FX_PDL"); c->cg_pdl = ev && ev[0] == '1'; }      // measured slower on B200: off unless asked for
    c->ready = true;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (int i = 0; i < 256; ++i) if (!g_all[i]) { g_all[i] = c; break; }
    }
    *out = c;
    return FX_OK;
}

extern "C" fx_status fx_create(fx_ctx** out, int32_t device, void* cuda_stream) {
    if (!out) { fx_set_error("fx_create: null pointer"); return FX_EINVAL; }
    return ctx_make(out, device, cuda_stream);
}
extern "C" void fx_destroy(fx_ctx* c) {
    if (!c) return;
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (int d = 0; d < FX_MAX_DEV; ++d) if (g_default[d] == c) g_default[d] = nullptr;
    }
    ctx_release(c);
}

FxCtx* fx_default_ctx() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= FX_MAX_DEV) {
        fx_set_error("no CUDA device: %s (libfx has no CPU fallback)", cudaGetErrorString(e));
        return nullptr;
    }
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_default[dev]) {
        FxCtx* c = nullptr;
        g_mu.unlock();                                      // ctx_make registers the context under the same mutex
        const fx_status s = ctx_make(&c, dev, nullptr);
        g_mu.lock();
        if (s != FX_OK) return nullptr;
        if (g_default[dev]) { g_mu.unlock(); ctx_release(c); g_mu.lock(); }       // another thread was faster
        else g_default[dev] = c;
    }
    return g_default[dev];
}

int fx_func_occ(FxCtx* c, const void* f, int block, size_t smem, bool carveout) {
    bool known = false;
    for (int i = 0; i < c->nfcache; ++i) {
        if (c->fcache[i].f != f) continue;
        known = true;
        if (c->fcache[i].block == block && c->fcache[i].smem == smem) return c->fcache[i].occ;
    }
    if (!known) {
        if (smem > 48 * 1024) cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (carveout) cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f, block, smem) != cudaSuccess || occ < 1) { occ = 1; cudaGetLastError(); }
    if (c->nfcache < (int)(sizeof(c->fcache) / sizeof(c->fcache[0]))) c->fcache[c->nfcache++] = {f, block, smem, occ};
    return occ;
}

extern "C" fx_status fx_set_stream_ex(fx_ctx* c, void* s) {
    FX_ENTER(c, "fx_set_stream");
    c->stream = (cudaStream_t)s;
    return FX_OK;
}
extern "C" fx_status fx_set_stream(void* s) { FxCtx* c = fx_default_ctx(); return c ? fx_set_stream_ex(c, s) : FX_ECUDA; }

extern "C" fx_status fx_set_launch_ex(fx_ctx* c, int32_t id, int32_t grid_dim, int32_t block_dim) {
    FX_ENTER(c, "fx_set_launch");
    if (id < 0 || id > 3 || grid_dim < 0 || block_dim < 0 || block_dim > 1024 || (block_dim & 31)) {
        fx_set_error("fx_set_launch: bad arguments"); return FX_EINVAL;
    }
    c->launch[id][0] = grid_dim; c->launch[id][1] = block_dim;
    return FX_OK;
}
extern "C" fx_status fx_set_launch(int32_t id, int32_t grid_dim, int32_t block_dim) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_set_launch_ex(c, id, grid_dim, block_dim) : FX_ECUDA;
}
extern "C" fx_status fx_set_cg_fused_ex(fx_ctx* c, int32_t fused) {
    FX_ENTER(c, "fx_set_cg_fused");
    if (fused < 0 || fused > 3) { fx_set_error("fx_set_cg_fused: mode must be 0..3"); return FX_EINVAL; }
    c->cg_fused = fused;
    return FX_OK;
}
extern "C" fx_status fx_set_cg_fused(int32_t fused) { FxCtx* c = fx_default_ctx(); return c ? fx_set_cg_fused_ex(c, fused) : FX_ECUDA; }
extern "C" fx_status fx_set_dg_path_ex(fx_ctx* c, int32_t path) {
    FX_ENTER(c, "fx_set_dg_path");
    if (path < 0 || path > 2) { fx_set_error("fx_set_dg_path: path must be 0..2"); return FX_EINVAL; }
    c->dg_path = path;
    return FX_OK;
}
extern "C" fx_status fx_set_dg_path(int32_t path) { FxCtx* c = fx_default_ctx(); return c ? fx_set_dg_path_ex(c, path) : FX_ECUDA; }

extern "C" fx_status fx_exdot_stats_ex(fx_ctx* c, uint64_t* out_host, int32_t reset) {
    FX_ENTER(c, "fx_exdot_stats");
    FX_CUDA(cudaStreamSynchronize(c->stream));
    if (out_host) FX_CUDA(cudaMemcpy(out_host, c->ex.stats, 4 * sizeof(fx_u64), cudaMemcpyDeviceToHost));
    if (reset) FX_CUDA(cudaMemset(c->ex.stats, 0, 4 * sizeof(fx_u64)));
    return FX_OK;
}
extern "C" fx_status fx_exdot_stats(uint64_t* out_host, int32_t reset) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_exdot_stats_ex(c, out_host, reset) : FX_ECUDA;
}

extern "C" int64_t fx_launch_count(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    long long n = g_launches_freed;
    for (int i = 0; i < 256; ++i) if (g_all[i]) n += g_all[i]->launches;
    return n;
}

// Releases the default contexts of all devices (contexts made by fx_create belong to their creators).
extern "C" void fx_shutdown(void) {
    FxCtx* d[FX_MAX_DEV];
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (int i = 0; i < FX_MAX_DEV; ++i) { d[i] = g_default[i]; g_default[i] = nullptr; }
    }
    for (int i = 0; i < FX_MAX_DEV; ++i) ctx_release(d[i]);
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

extern "C" fx_status fx_axpby_ex(fx_ctx* c, double alpha, const double* x, double beta, double* y, int64_t n) {
    FX_ENTER(c, "fx_axpby");
    if (n < 0 || (n > 0 && (!x || !y))) { fx_set_error("fx_axpby: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    const bool vec = aligned16(x) && aligned16(y);
    int grid, block; ew_shape(c, n, vec, &grid, &block);
    if (beta == 0.0) { if (vec) k_axpby<true, true><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); else k_axpby<true, false><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); }
    else { if (vec) k_axpby<false, true><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); else k_axpby<false, false><<<grid, block, 0, c->stream>>>(alpha, x, beta, y, n); }
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}
extern "C" fx_status fx_axpby(double alpha, const double* x, double beta, double* y, int64_t n) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_axpby_ex(c, alpha, x, beta, y, n) : FX_ECUDA;
}

extern "C" fx_status fx_pointwise_dot_ex(fx_ctx* c, double alpha, const double* x1, const double* x2, double beta, double* y, int64_t n) {
    FX_ENTER(c, "fx_pointwise_dot");
    if (n < 0 || (n > 0 && (!x1 || !x2 || !y))) { fx_set_error("fx_pointwise_dot: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    const bool vec = aligned16(x1) && aligned16(x2) && aligned16(y);
    int grid, block; ew_shape(c, n, vec, &grid, &block);
    if (beta == 0.0) { if (vec) k_pointwise<true, true><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); else k_pointwise<true, false><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); }
    else { if (vec) k_pointwise<false, true><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); else k_pointwise<false, false><<<grid, block, 0, c->stream>>>(alpha, x1, x2, beta, y, n); }
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}
extern "C" fx_status fx_pointwise_dot(double alpha, const double* x1, const double* x2, double beta, double* y, int64_t n) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_pointwise_dot_ex(c, alpha, x1, x2, beta, y, n) : FX_ECUDA;
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

extern "C" fx_status fx_pointwise_dot2_ex(fx_ctx* c, double alpha, const double* x1, const double* y1, double beta, const double* x2, const double* y2,
                                       double gamma, double* z, int64_t n) {
    FX_ENTER(c, "fx_pointwise_dot2");
    if (n < 0 || (n > 0 && (!x1 || !y1 || !x2 || !y2 || !z))) { fx_set_error("fx_pointwise_dot2: bad arguments"); return FX_EINVAL; }
    if (n == 0) return FX_OK;
    int grid, block; ew_shape(c, n, false, &grid, &block);
    if (gamma == 0.0) k_pointwise2<true><<<grid, block, 0, c->stream>>>(alpha, x1, y1, beta, x2, y2, gamma, z, n);
    else k_pointwise2<false><<<grid, block, 0, c->stream>>>(alpha, x1, y1, beta, x2, y2, gamma, z, n);
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}
extern "C" fx_status fx_pointwise_dot2(double alpha, const double* x1, const double* y1, double beta, const double* x2, const double* y2,
                                       double gamma, double* z, int64_t n) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_pointwise_dot2_ex(c, alpha, x1, y1, beta, x2, y2, gamma, z, n) : FX_ECUDA;
}
