// fx_ops.cu -- exact-dot kernel, dG apply kernel, dG weights, and their C ABI entry points (include/fx.h).

#include <math.h>
#include <string.h>

#include <mutex>

#include "fx_internal.h"
#include "fx_dgt.cuh"
#include "fx_stream.cuh"

// ------------------------------------------------------------------------------------------------------------
// exact dot  (design in fx_exdot.cuh / DESIGN.md 6.1).  HBM roofline: 16 B per element.
// ------------------------------------------------------------------------------------------------------------

#define EX_K 4
#define EX_W 40
#ifndef EX_KL
#define EX_KL 2            // low window of the stand-alone reductions (fx_exdot.cuh): 6 x 40 = 240 bit before the long accumulator
#endif
typedef ExAcc<EX_K, EX_W, EX_KL> ExDotAcc;
#define EX_U 4
#define EX_STAGES 4

// Tiles of blockDim.x * EX_U elements, grid-stride; FX_STAGES-1 tiles in flight per thread through cp.async.
// Shared layout (doubles): [stage][array 0..1][u][thread]   (VEC: [stage][array][u/2][thread] of 16 B)
template <bool VEC>
__device__ __forceinline__ void exdot_issue(double* buf, int stage, const double* __restrict__ x, const double* __restrict__ y,
                                            long long n, long long base, bool live) {
    const int bd = blockDim.x;
    double* sx = buf + (size_t)stage * 2 * EX_U * bd;
    double* sy = sx + EX_U * bd;
    FX_ASSERT(stage >= 0 && stage < EX_STAGES && base >= 0 && (!live || base < n + (long long)EX_U * bd));
    if (live) {
        if (VEC) {
#pragma unroll
            for (int u = 0; u < EX_U / 2; ++u) {
                const int slot = 2 * (u * bd + threadIdx.x);
                const long long e0 = base + slot;
                const long long left = n - e0;
                const int bytes = left >= 2 ? 16 : (left == 1 ? 8 : 0);
                const long long es = bytes ? e0 : 0;                 // keep the address valid when nothing is copied
                fx_cp_async16(fx_smem_addr(sx + slot), x + es, bytes);
                fx_cp_async16(fx_smem_addr(sy + slot), y + es, bytes);
            }
        } else {
#pragma unroll
            for (int u = 0; u < EX_U; ++u) {
                const int slot = u * bd + threadIdx.x;
                const long long e0 = base + slot;
                const bool in = e0 < n;
                fx_cp_async8(fx_smem_addr(sx + slot), x + (in ? e0 : 0), in);
                fx_cp_async8(fx_smem_addr(sy + slot), y + (in ? e0 : 0), in);
            }
        }
    }
    fx_cp_commit();
}

// Consume one landed tile from shared memory (generic: bounds-checked).
// MODE 1 (sum): the two arrays are the two halves of one vector whose exact sum is wanted -- every element is accumulated
// as element * 1 (no error term); same loads, same ring, about the same fp64 work per byte as the dot.
// MODE 2 (binary32 dot): every 8-byte slot holds two floats; float * float is exact in fp64 (no error term).
template <int MODE>
__device__ __forceinline__ void ex_feed(ExDotAcc& acc, const double (&xv)[EX_U], const double (&yv)[EX_U], const bool (&act)[EX_U],
                                        ExShared* sh) {
    if (MODE == 1) {
        double one[EX_U];
#pragma unroll
        for (int u = 0; u < EX_U; ++u) one[u] = 1.0;
        acc.add<EX_U, false, true>(xv, one, act, sh);
        acc.add<EX_U, false, true>(yv, one, act, sh);
    } else if (MODE == 2) {
        double a[2 * EX_U], b[2 * EX_U];
        bool ac[2 * EX_U];
#pragma unroll
        for (int u = 0; u < EX_U; ++u) {
            a[2 * u] = __int_as_float(__double2loint(xv[u])); a[2 * u + 1] = __int_as_float(__double2hiint(xv[u]));
            b[2 * u] = __int_as_float(__double2loint(yv[u])); b[2 * u + 1] = __int_as_float(__double2hiint(yv[u]));
            ac[2 * u] = act[u]; ac[2 * u + 1] = act[u];
        }
        acc.add<2 * EX_U, false, true>(a, b, ac, sh);
    } else acc.add<EX_U>(xv, yv, act, sh);
}

// the same for a full tile (the hot loop): no activity flags, and the 2 * EX_U values of the sum as ONE batch (one range test
// and one branch per 8 values instead of two batches with selects: the sum is issue-bound; 5.3 -> 5.9 TB/s at 2^26)
template <int MODE>
__device__ __forceinline__ void ex_feed_full(ExDotAcc& acc, const double (&xv)[EX_U], const double (&yv)[EX_U], ExShared* sh) {
    if (MODE == 1) {
        double v[2 * EX_U], one[2 * EX_U];
        bool all[2 * EX_U];
#pragma unroll
        for (int u = 0; u < EX_U; ++u) { v[u] = xv[u]; v[EX_U + u] = yv[u]; one[u] = 1.0; one[EX_U + u] = 1.0; all[u] = true; all[EX_U + u] = true; }
        acc.add<2 * EX_U, true, true>(v, one, all, sh);
    } else if (MODE == 2) {                                          // (the binary32 dot measured 2 % slower as one flag-free batch)
        bool act[EX_U];
#pragma unroll
        for (int u = 0; u < EX_U; ++u) act[u] = true;
        ex_feed<2>(acc, xv, yv, act, sh);
    } else acc.add_all<EX_U>(xv, yv, sh);
}

template <bool VEC, int MODE>
__device__ __forceinline__ void exdot_consume(const double* buf, int stage, long long n, long long base, ExDotAcc& acc,
                                              ExShared* sh) {
    const int bd = blockDim.x;
    const double* sx = buf + (size_t)stage * 2 * EX_U * bd;
    const double* sy = sx + EX_U * bd;
    double xv[EX_U], yv[EX_U];
    bool act[EX_U];
    if (VEC) {
#pragma unroll
        for (int u = 0; u < EX_U / 2; ++u) {
            const int slot = 2 * (u * bd + threadIdx.x);
            const double2 a = *reinterpret_cast<const double2*>(sx + slot);
            const double2 b = *reinterpret_cast<const double2*>(sy + slot);
            xv[2 * u] = a.x; xv[2 * u + 1] = a.y; yv[2 * u] = b.x; yv[2 * u + 1] = b.y;
            act[2 * u] = base + slot < n; act[2 * u + 1] = base + slot + 1 < n;
        }
    } else {
#pragma unroll
        for (int u = 0; u < EX_U; ++u) {
            const int slot = u * bd + threadIdx.x;
            xv[u] = sx[slot]; yv[u] = sy[slot];
            act[u] = base + slot < n;
        }
    }
    ex_feed<MODE>(acc, xv, yv, act, sh);
}

// The kernel.  CTA b takes tiles b, b+G, b+2G, ...; EX_STAGES-1 tiles are in flight per thread.
// Hot loop (16-byte aligned inputs, full tiles): pointer increments only, compile-time stage offsets, no bounds.
template <bool VEC, int MODE>
__global__ void __launch_bounds__(256, 2) k_exdot(const double* __restrict__ x, const double* __restrict__ y, long long n,
                                                  ExGlobal g, int first, int last, double* result) {
    extern __shared__ __align__(16) double ex_buf[];
    __shared__ ExShared sh;
    ex_shared_init(&sh);
    ExDotAcc acc;
    acc.init();
    const int bd = blockDim.x;
    const long long tile = (long long)bd * EX_U;
    const long long ntiles = (n + tile - 1) / tile, nfull = n / tile;
    long long tq = blockIdx.x;                                   // next tile to issue
    long long t = blockIdx.x;                                    // next tile to consume
#pragma unroll
    for (int s = 0; s < EX_STAGES - 1; ++s) { exdot_issue<VEC>(ex_buf, s, x, y, n, tq * tile, tq < ntiles); tq += gridDim.x; }
    int stage = 0;
    if (VEC) {
        // per-thread pointers of the tile to issue; shared slots of this thread
        const long long step = (long long)gridDim.x * tile;
        const double* gx = x + tq * tile + 2 * threadIdx.x;
        const double* gy = y + tq * tile + 2 * threadIdx.x;
        const unsigned s0 = fx_smem_addr(ex_buf) + 16u * threadIdx.x;
        const unsigned stage_bytes = 2u * EX_U * bd * 8u, arr_bytes = (unsigned)EX_U * bd * 8u, u_bytes = 16u * bd;
        unsigned so = 0;                                             // byte offset of the stage to consume
        unsigned sqo = (EX_STAGES - 1) * stage_bytes;                // ... and of the stage to fill
        // number of hot iterations as a 32-bit down-counter; pointers are kept as opaque induction variables (the
        // empty asm stops the compiler from re-deriving them from the tile index with 64-bit multiplies every iteration)
        int hot = tq < nfull ? (int)((nfull - tq + gridDim.x - 1) / gridDim.x) : 0;
        tq += (long long)hot * gridDim.x; t += (long long)hot * gridDim.x;
        for (; hot > 0; --hot) {                                     // the tile to issue is a full one
#pragma unroll
            for (int u = 0; u < EX_U / 2; ++u) {
                fx_cp_async16_full(s0 + sqo + u * u_bytes, gx + 2 * u * bd);
                fx_cp_async16_full(s0 + sqo + arr_bytes + u * u_bytes, gy + 2 * u * bd);
            }
            fx_cp_commit();
            gx += step; gy += step;
            asm volatile("" : "+l"(gx), "+l"(gy));
            fx_cp_wait<EX_STAGES - 1>();
            double xv[EX_U], yv[EX_U];
#pragma unroll
            for (int u = 0; u < EX_U / 2; ++u) {
                double2 a, b;
                fx_lds128(a, s0 + so + u * u_bytes);
                fx_lds128(b, s0 + so + arr_bytes + u * u_bytes);
                xv[2 * u] = a.x; xv[2 * u + 1] = a.y; yv[2 * u] = b.x; yv[2 * u + 1] = b.y;
            }
            ex_feed_full<MODE>(acc, xv, yv, &sh);                    // consumed tile < issued tile: full as well
            sqo = so;
            so += stage_bytes; if (so == EX_STAGES * stage_bytes) so = 0;
            if (++stage == EX_STAGES) stage = 0;
        }
    }
    for (; t < ntiles; t += gridDim.x) {                                     // generic: tail tiles, unaligned inputs
        int sq = stage + EX_STAGES - 1; if (sq >= EX_STAGES) sq -= EX_STAGES;
        exdot_issue<VEC>(ex_buf, sq, x, y, n, tq * tile, tq < ntiles); tq += gridDim.x;
        fx_cp_wait<EX_STAGES - 1>();
        exdot_consume<VEC, MODE>(ex_buf, stage, n, t * tile, acc, &sh);
        if (++stage == EX_STAGES) stage = 0;
    }
    fx_cp_wait<0>();
#if defined(FX_EX_SKIP) && FX_EX_SKIP == 1
    if (n == -12345) { acc.flush(&sh); ex_block_finish(&sh, g, first, last, result); }
#elif defined(FX_EX_SKIP) && FX_EX_SKIP == 2
    acc.flush(&sh);
    if (n == -12345) ex_block_finish(&sh, g, first, last, result);
#else
    acc.flush(&sh);
    ex_block_finish(&sh, g, first, last, result);
#endif
}

// one launch over m <= 2^28 elements (keeps every 64-bit digit far from overflow); first/last: position in the call
fx_status fx_launch_exdot_part(FxCtx* c, const double* x, const double* y, int64_t m, int first, int last, double* result_dev, int mode) {
    const bool vec = aligned16(x) && aligned16(y);
    int bd = c->launch[0][1] ? c->launch[0][1] : 256;
    if (bd > 256) bd = 256;                     // compiled for <= 256 threads per CTA
    const size_t smem = (size_t)EX_STAGES * 2 * EX_U * bd * sizeof(double);
    // (the six instantiations share one shared-memory layout: the dynamic limit is raised for the one that is launched)
    const void* kf = mode == 1 ? (vec ? (const void*)k_exdot<true, 1> : (const void*)k_exdot<false, 1>)
                   : mode == 2 ? (vec ? (const void*)k_exdot<true, 2> : (const void*)k_exdot<false, 2>)
                               : (vec ? (const void*)k_exdot<true, 0> : (const void*)k_exdot<false, 0>);
    const int occ = fx_func_occ(c, kf, bd, smem);
    const long long tile = (long long)bd * EX_U;
    long long grid = (m + tile - 1) / tile;
    const long long gmax = (long long)c->num_sms * occ;             // one resident wave: every CTA pays one flush + merge
    if (grid > gmax) grid = gmax;
    if (grid <= EX_STAGES) grid = 1;                                 // a few tiles: one CTA has them all in flight at once and finishes
    if (grid < 1) grid = 1;                                          // alone -- no digit round trips through L2, no ticket (6 us against 8)
    if (c->launch[0][0]) grid = c->launch[0][0];
#define FX_EXDOT_GO(M) \
    if (vec) k_exdot<true, M><<<(int)grid, bd, smem, c->stream>>>(x, y, m, c->ex, first, last, result_dev); \
    else k_exdot<false, M><<<(int)grid, bd, smem, c->stream>>>(x, y, m, c->ex, first, last, result_dev);
    if (mode == 1) { FX_EXDOT_GO(1) } else if (mode == 2) { FX_EXDOT_GO(2) } else { FX_EXDOT_GO(0) }
#undef FX_EXDOT_GO
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

// ---- weighted dot (NA = 3: x, w, y) and exact sum (NA = 1) -- SURVEY 8f-3 ---------------------------------------------
// Same accumulator, same single-pass finaliser; generic cp.async ring (8-byte copies: no alignment requirement).
template <int NA, bool VEC>
__global__ void __launch_bounds__(256, 2) k_exdotn(const double* __restrict__ a0, const double* __restrict__ a1,
                                                   const double* __restrict__ a2, long long n, ExGlobal g, int first, int last,
                                                   double* result) {
    extern __shared__ __align__(16) double ex_buf[];
    __shared__ ExShared sh;
    ex_shared_init(&sh);
    ExDotAcc acc;
    acc.init();
    const int bd = blockDim.x;
    const long long tile = (long long)bd * EX_U, ntiles = (n + tile - 1) / tile;
    const double* arr[3] = {a0, a1, a2};
    auto issue = [&](int stage, long long t) {
        double* s0 = ex_buf + (size_t)stage * NA * EX_U * bd;
        if (t < ntiles) {
            if (VEC) {                                               // 16-byte copies: all arrays 16-byte aligned
#pragma unroll
                for (int u = 0; u < EX_U / 2; ++u) {
                    const int slot = 2 * (u * bd + threadIdx.x);
                    const long long e = t * tile + slot;
                    const long long left = n - e;
                    const int bytes = left >= 2 ? 16 : (left == 1 ? 8 : 0);
#pragma unroll
                    for (int a = 0; a < NA; ++a) fx_cp_async16(fx_smem_addr(s0 + a * EX_U * bd + slot), arr[a] + (bytes ? e : 0), bytes);
                }
            } else {
#pragma unroll
                for (int u = 0; u < EX_U; ++u) {
                    const int slot = u * bd + threadIdx.x;
                    const long long e = t * tile + slot;
                    const bool in = e < n;
#pragma unroll
                    for (int a = 0; a < NA; ++a) fx_cp_async8(fx_smem_addr(s0 + a * EX_U * bd + slot), arr[a] + (in ? e : 0), in);
                }
            }
        }
        fx_cp_commit();
    };
    long long tq = blockIdx.x;
#pragma unroll
    for (int s = 0; s < EX_STAGES - 1; ++s) { issue(s, tq); tq += gridDim.x; }
    int stage = 0;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int sq = stage + EX_STAGES - 1; if (sq >= EX_STAGES) sq -= EX_STAGES;
        issue(sq, tq); tq += gridDim.x;
        fx_cp_wait<EX_STAGES - 1>();
        const double* s0 = ex_buf + (size_t)stage * NA * EX_U * bd;
        double xv[EX_U], yv[EX_U];
        bool act[EX_U];
        if (VEC) {
#pragma unroll
            for (int u = 0; u < EX_U / 2; ++u) {
                const int slot = 2 * (u * bd + threadIdx.x);
                act[2 * u] = t * tile + slot < n; act[2 * u + 1] = t * tile + slot + 1 < n;
                const double2 a = *reinterpret_cast<const double2*>(s0 + slot);
                if (NA == 3) {
                    const double2 w = *reinterpret_cast<const double2*>(s0 + EX_U * bd + slot);
                    const double2 b = *reinterpret_cast<const double2*>(s0 + 2 * EX_U * bd + slot);
                    xv[2 * u] = __dmul_rn(a.x, w.x); xv[2 * u + 1] = __dmul_rn(a.y, w.y); yv[2 * u] = b.x; yv[2 * u + 1] = b.y;
                } else { xv[2 * u] = a.x; xv[2 * u + 1] = a.y; yv[2 * u] = act[2 * u] ? 1.0 : 0.0; yv[2 * u + 1] = act[2 * u + 1] ? 1.0 : 0.0; }
            }
        } else {
#pragma unroll
            for (int u = 0; u < EX_U; ++u) {
                const int slot = u * bd + threadIdx.x;
                act[u] = t * tile + slot < n;
                if (NA == 3) { xv[u] = __dmul_rn(s0[slot], s0[EX_U * bd + slot]); yv[u] = s0[2 * EX_U * bd + slot]; }   // u = RN(x*w)
                else { xv[u] = s0[slot]; yv[u] = act[u] ? 1.0 : 0.0; }
            }
        }
        if (NA == 1) acc.add<EX_U, false, true>(xv, yv, act, &sh);   // x * 1 is exact: no error term
        else if (VEC && (t + 1) * tile <= n) acc.add_all<EX_U>(xv, yv, &sh);   // full tile: no activity flags
        else acc.add<EX_U>(xv, yv, act, &sh);
        if (++stage == EX_STAGES) stage = 0;
    }
    fx_cp_wait<0>();
    acc.flush(&sh);
    ex_block_finish(&sh, g, first, last, result);
}

template <int NA>
static fx_status launch_exdotn(FxCtx* c, const double* a0, const double* a1, const double* a2, int64_t n, double* result_dev) {
    const int bd = 256;
    const size_t smem = (size_t)EX_STAGES * NA * EX_U * bd * sizeof(double);
    const int occ = fx_func_occ(c, (const void*)k_exdotn<NA, true>, bd, smem);
    fx_func_occ(c, (const void*)k_exdotn<NA, false>, bd, smem);
    const int64_t CHUNK = (int64_t)1 << 28;
    int64_t done = 0;
    do {
        const int64_t m = (n - done < CHUNK) ? (n - done) : CHUNK;
        const long long tile = (long long)bd * EX_U;
        long long grid = (m + tile - 1) / tile;
        if (grid > (long long)c->num_sms * occ) grid = (long long)c->num_sms * occ;
        if (grid < 1) grid = 1;
        const bool vec = aligned16(a0) && (!a1 || aligned16(a1)) && (!a2 || aligned16(a2));     // (done is a multiple of 2^28)
        if (vec) k_exdotn<NA, true><<<(int)grid, bd, smem, c->stream>>>(a0 + done, a1 ? a1 + done : nullptr, a2 ? a2 + done : nullptr, m, c->ex,
                                                                        done == 0, done + m == n, result_dev);
        else k_exdotn<NA, false><<<(int)grid, bd, smem, c->stream>>>(a0 + done, a1 ? a1 + done : nullptr, a2 ? a2 + done : nullptr, m, c->ex,
                                                                     done == 0, done + m == n, result_dev);
        c->launches++;
        FX_CUDA(cudaGetLastError());
        done += m;
    } while (done < n);
    return FX_OK;
}

// ---- binary32 inputs, exact accumulation ---------------------------------------------------------------------
// Every product of two floats is exact in fp64 (48-bit mantissa), so p = (double)x * (double)y carries no error term
// (NOERR path: 3K fp64 operations per element).  8 elements per thread and tile; 16-byte cp.async when both arrays are
// 16-byte aligned, 4-byte copies otherwise.
#define EXF_U 8
template <bool VEC>
__global__ void __launch_bounds__(256, 2) k_exdot_f32(const float* __restrict__ x, const float* __restrict__ y, long long n, ExGlobal g,
                                                       int first, int last, double* result) {
    extern __shared__ __align__(16) float exf_buf[];
    __shared__ ExShared sh;
    ex_shared_init(&sh);
    ExDotAcc acc;
    acc.init();
    const int bd = blockDim.x;
    const long long tile = (long long)bd * EXF_U, ntiles = (n + tile - 1) / tile;
    auto issue = [&](int stage, long long t) {
        float* sx = exf_buf + (size_t)stage * 2 * EXF_U * bd;
        float* sy = sx + EXF_U * bd;
        if (t < ntiles) {
            if (VEC) {
#pragma unroll
                for (int u = 0; u < EXF_U / 4; ++u) {
                    const int slot = 4 * (u * bd + threadIdx.x);
                    const long long e = t * tile + slot, left = n - e;
                    const int bytes = left >= 4 ? 16 : (left > 0 ? 4 * (int)left : 0);
                    const long long es = bytes ? e : 0;
                    fx_cp_async16(fx_smem_addr(sx + slot), x + es, bytes);
                    fx_cp_async16(fx_smem_addr(sy + slot), y + es, bytes);
                }
            } else {
#pragma unroll
                for (int u = 0; u < EXF_U; ++u) {
                    const int slot = u * bd + threadIdx.x;
                    const long long e = t * tile + slot;
                    const bool in = e < n;
                    fx_cp_async4(fx_smem_addr(sx + slot), x + (in ? e : 0), in);
                    fx_cp_async4(fx_smem_addr(sy + slot), y + (in ? e : 0), in);
                }
            }
        }
        fx_cp_commit();
    };
    long long tq = blockIdx.x;
#pragma unroll
    for (int s = 0; s < EX_STAGES - 1; ++s) { issue(s, tq); tq += gridDim.x; }
    int stage = 0;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int sq = stage + EX_STAGES - 1; if (sq >= EX_STAGES) sq -= EX_STAGES;
        issue(sq, tq); tq += gridDim.x;
        fx_cp_wait<EX_STAGES - 1>();
        const float* sx = exf_buf + (size_t)stage * 2 * EXF_U * bd;
        const float* sy = sx + EXF_U * bd;
        double xv[EXF_U], yv[EXF_U];
        bool act[EXF_U];
        if (VEC) {
#pragma unroll
            for (int u = 0; u < EXF_U / 4; ++u) {
                const int slot = 4 * (u * bd + threadIdx.x);
                const float4 a = *reinterpret_cast<const float4*>(sx + slot), b = *reinterpret_cast<const float4*>(sy + slot);
                const long long e = t * tile + slot;
                xv[4 * u] = a.x; xv[4 * u + 1] = a.y; xv[4 * u + 2] = a.z; xv[4 * u + 3] = a.w;
                yv[4 * u] = b.x; yv[4 * u + 1] = b.y; yv[4 * u + 2] = b.z; yv[4 * u + 3] = b.w;
#pragma unroll
                for (int i = 0; i < 4; ++i) act[4 * u + i] = e + i < n;
            }
        } else {
#pragma unroll
            for (int u = 0; u < EXF_U; ++u) {
                const int slot = u * bd + threadIdx.x;
                xv[u] = sx[slot]; yv[u] = sy[slot];
                act[u] = t * tile + slot < n;
            }
        }
        acc.add<EXF_U, false, true>(xv, yv, act, &sh);                 // float * float is exact in fp64: no error term
        if (++stage == EX_STAGES) stage = 0;
    }
    fx_cp_wait<0>();
    acc.flush(&sh);
    ex_block_finish(&sh, g, first, last, result);
}

// result_host: host double (synchronises)
extern "C" fx_status fx_exdot_f32_ex(fx_ctx* c, const float* x, const float* y, int64_t n, double* result_host) {
    FX_ENTER(c, "fx_exdot_f32");
    if (n < 0 || (n > 0 && (!x || !y)) || !result_host) { fx_set_error("fx_exdot_f32: bad arguments"); return FX_EINVAL; }
    const int bd = 256;
    const size_t smem = (size_t)EX_STAGES * 2 * EXF_U * bd * sizeof(float);
    const int occ = fx_func_occ(c, (const void*)k_exdot_f32<true>, bd, smem);
    fx_func_occ(c, (const void*)k_exdot_f32<false>, bd, smem);
    const bool vec = aligned16(x) && aligned16(y);
    const int64_t CHUNK = (int64_t)1 << 28;
    int64_t done = 0;
    // long, 8-byte aligned inputs: pairs of floats through the fp64 dot kernel's ring (k_exdot<., 2>), 2^27 pairs per
    // launch; an odd last element (or short / 4-byte aligned input) through the generic kernel below
    if (n >= 8192 && ((uintptr_t)x & 7) == 0 && ((uintptr_t)y & 7) == 0) {
        const int64_t SLOTS = (int64_t)1 << 27;
        while (n - done >= 2) {
            int64_t h = (n - done) / 2;
            if (h > SLOTS) h = SLOTS;
            const fx_status sp = fx_launch_exdot_part(c, (const double*)(x + done), (const double*)(y + done), h, done == 0, done + 2 * h == n, c->result_dev, 2);
            if (sp != FX_OK) return sp;
            done += 2 * h;
        }
    }
    const bool tailvec = vec && done == 0;
    if (done < n || n == 0) do {
        const int64_t m = (n - done < CHUNK) ? (n - done) : CHUNK;
        const long long tile = (long long)bd * EXF_U;
        long long grid = (m + tile - 1) / tile;
        if (grid > (long long)c->num_sms * occ) grid = (long long)c->num_sms * occ;
        if (grid < 1) grid = 1;
        if (tailvec) k_exdot_f32<true><<<(int)grid, bd, smem, c->stream>>>(x + done, y + done, m, c->ex, done == 0, done + m == n, c->result_dev);
        else k_exdot_f32<false><<<(int)grid, bd, smem, c->stream>>>(x + done, y + done, m, c->ex, done == 0, done + m == n, c->result_dev);
        c->launches++;
        FX_CUDA(cudaGetLastError());
        done += m;
    } while (done < n);
    return fx_result_to_host(c, result_host);
}
// the plain-named reductions return the value; NaN with a non-empty fx_last_error() is a failure, with an empty one a genuine NaN
#define FX_PLAIN_VALUE(call)                        \
    fx_set_error("%s", "");                         \
    FxCtx* c = fx_default_ctx();                    \
    if (!c) return NAN;                             \
    double v = NAN;                                 \
    return (call) == FX_OK ? v : NAN;
extern "C" double fx_exdot_f32(const float* x, const float* y, int64_t n) { FX_PLAIN_VALUE(fx_exdot_f32_ex(c, x, y, n, &v)) }

// the double a finished reduction left in the context's device slot -> host (synchronises)
fx_status fx_result_to_host(FxCtx* c, double* result_host) {
    FX_CUDA(cudaMemcpyAsync(c->result_pinned, c->result_dev, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    FX_CUDA(cudaStreamSynchronize(c->stream));
    *result_host = c->result_pinned[0];
    return FX_OK;
}

extern "C" fx_status fx_exdot3_ex(fx_ctx* c, const double* x, const double* w, const double* y, int64_t n, double* result_host) {
    FX_ENTER(c, "fx_exdot3");
    if (n < 0 || (n > 0 && (!x || !w || !y)) || !result_host) { fx_set_error("fx_exdot3: bad arguments"); return FX_EINVAL; }
    const fx_status s = launch_exdotn<3>(c, x, w, y, n, c->result_dev);
    return s != FX_OK ? s : fx_result_to_host(c, result_host);
}
extern "C" double fx_exdot3(const double* x, const double* w, const double* y, int64_t n) { FX_PLAIN_VALUE(fx_exdot3_ex(c, x, w, y, n, &v)) }

// Exact sum: long vectors go through the dot kernel's ring as two halves (x[0,h) and x[h,2h), h even so that both keep
// the alignment of x), 2^27 elements per half and launch; what is left (<= 3 elements, or a short vector) through the
// generic kernel.  All launches accumulate into the same digits; the last one rounds.
fx_status fx_launch_exsum(FxCtx* c, const double* x, int64_t n, double* result_dev) {
    if (n < 4096) return launch_exdotn<1>(c, x, nullptr, nullptr, n, result_dev);
    const int64_t HALF = (int64_t)1 << 27;
    int64_t done = 0;
    bool first = true;
    while (n - done >= 4) {
        int64_t h = ((n - done) / 2) & ~(int64_t)1;
        if (h > HALF) h = HALF;
        const bool last = done + 2 * h == n;
        fx_status s = fx_launch_exdot_part(c, x + done, x + done + h, h, first, last, result_dev, 1);
        if (s != FX_OK) return s;
        first = false;
        done += 2 * h;
    }
    if (done < n) {
        k_exdotn<1, false><<<1, 256, (size_t)EX_STAGES * EX_U * 256 * sizeof(double), c->stream>>>(x + done, nullptr, nullptr, n - done, c->ex, 0, 1, result_dev);
        c->launches++;
        FX_CUDA(cudaGetLastError());
    }
    return FX_OK;
}

extern "C" fx_status fx_exsum_ex(fx_ctx* c, const double* x, int64_t n, double* result_host) {
    FX_ENTER(c, "fx_exsum");
    if (n < 0 || (n > 0 && !x) || !result_host) { fx_set_error("fx_exsum: bad arguments"); return FX_EINVAL; }
    const fx_status s = fx_launch_exsum(c, x, n, c->result_dev);
    return s != FX_OK ? s : fx_result_to_host(c, result_host);
}
extern "C" double fx_exsum(const double* x, int64_t n) { FX_PLAIN_VALUE(fx_exsum_ex(c, x, n, &v)) }

fx_status fx_launch_exdot(FxCtx* c, const double* x, const double* y, int64_t n, double* result_dev) {
    const int64_t CHUNK = (int64_t)1 << 28;
    int64_t done = 0;
    do {
        const int64_t m = (n - done < CHUNK) ? (n - done) : CHUNK;
        fx_status s = fx_launch_exdot_part(c, x + done, y + done, m, done == 0, done + m == n, result_dev);
        if (s != FX_OK) return s;
        done += m;
    } while (done < n);
    return FX_OK;
}

extern "C" fx_status fx_exdot_async_ex(fx_ctx* c, const double* x, const double* y, int64_t n, double* result_dev) {
    FX_ENTER(c, "fx_exdot_async");
    if (n < 0 || (n > 0 && (!x || !y)) || !result_dev) { fx_set_error("fx_exdot_async: bad arguments"); return FX_EINVAL; }
    return fx_launch_exdot(c, x, y, n, result_dev);
}
extern "C" fx_status fx_exdot_async(const double* x, const double* y, int64_t n, double* result_dev) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_exdot_async_ex(c, x, y, n, result_dev) : FX_ECUDA;
}

// result_host (host double, synchronises) and/or result_dev (device double, stream-ordered); at least one
extern "C" fx_status fx_exdot_ex(fx_ctx* c, const double* x, const double* y, int64_t n, double* result_host, double* result_dev) {
    FX_ENTER(c, "fx_exdot");
    if (n < 0 || (n > 0 && (!x || !y)) || (!result_host && !result_dev)) { fx_set_error("fx_exdot: bad arguments"); return FX_EINVAL; }
    fx_status s = fx_launch_exdot(c, x, y, n, c->result_dev);
    if (s != FX_OK) return s;
    if (result_dev) FX_CUDA(cudaMemcpyAsync(result_dev, c->result_dev, sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    return result_host ? fx_result_to_host(c, result_host) : FX_OK;
}
extern "C" double fx_exdot(const double* x, const double* y, int64_t n) { FX_PLAIN_VALUE(fx_exdot_ex(c, x, y, n, &v, nullptr)) }

extern "C" fx_status fx_exdot_digits_ex(fx_ctx* c, const double* x, const double* y, int64_t n, uint64_t* limbs_host, int32_t* flags_host,
                                     double* result_host) {
    FX_ENTER(c, "fx_exdot_digits");
    if (n < 0 || (n > 0 && (!x || !y)) || !limbs_host) { fx_set_error("fx_exdot_digits: bad arguments"); return FX_EINVAL; }
    // flags are cleared by the finaliser after rounding; read them through the result instead: launch, then copy
    c->ex.keep_limbs = 1;                      // (a plain dot does not write the canonical limbs back)
    fx_status s = fx_launch_exdot(c, x, y, n, c->result_dev);
    c->ex.keep_limbs = 0;
    if (s != FX_OK) return s;
    FX_CUDA(cudaStreamSynchronize(c->stream));
    FX_CUDA(cudaMemcpy(limbs_host, c->ex.limbs, FX_NLIMB * sizeof(fx_u64), cudaMemcpyDeviceToHost));
    int fl[2] = {0, 0};
    FX_CUDA(cudaMemcpy(fl, c->ex.flags, 2 * sizeof(int), cudaMemcpyDeviceToHost));
    if (flags_host) { flags_host[0] = (fl[1] & FX_FLAG_NAN) != 0; flags_host[1] = (fl[1] & FX_FLAG_PINF) != 0; flags_host[2] = (fl[1] & FX_FLAG_NINF) != 0; }
    if (result_host) FX_CUDA(cudaMemcpy(result_host, c->result_dev, sizeof(double), cudaMemcpyDeviceToHost));
    return FX_OK;
}
extern "C" fx_status fx_exdot_digits(const double* x, const double* y, int64_t n, uint64_t* limbs_host, int32_t* flags_host,
                                     double* result_host) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_exdot_digits_ex(c, x, y, n, limbs_host, flags_host, result_host) : FX_ECUDA;
}

// ------------------------------------------------------------------------------------------------------------
// dG elliptic apply  (fx_dg.cuh / DESIGN.md 6.2).  HBM roofline: 24 B per unknown.
// ------------------------------------------------------------------------------------------------------------

struct NoAcc {
    template <int U> __device__ void add(const double (&)[U], const double (&)[U], const bool (&)[U], ExShared*) {}
    template <int U> __device__ void add_all(const double (&)[U], const double (&)[U], ExShared*) {}
};

#ifndef FX_AP_R
#define FX_AP_R 168      // registers per thread / warps per CTA of k_dg_apply<3>
#define FX_AP_W 4
#endif
template <int P, bool NEU>
__global__ void __maxnreg__(P <= 2 ? 128 : P == 3 ? FX_AP_R : 255) k_dg_apply(const __grid_constant__ DgParams g, const double* __restrict__ chi,
                                                  const double* __restrict__ x, double* __restrict__ y) {
    const int wpb = blockDim.x >> 5;
    long long w = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    const long long per = (long long)g.nstrip * g.nseg;                       // warps per plane
    if (w >= per * g.Nz) return;
    const long long zoff = (w / per) * ((long long)g.Nx * g.Ny * P * P);      // 3-D product grid: this warp's plane
    w %= per;
    chi += zoff; x += zoff; y += zoff;
    // consecutive warps take consecutive strips of the same row segment: neighbouring halo columns are L1/L2 hits
    const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);
    const int j0 = seg * g.rows_per_seg;
    int j1 = j0 + g.rows_per_seg;
    if (j1 > g.Ny) j1 = g.Ny;
    const DgSrc src = {x, nullptr, nullptr, 0.0, false};
    extern __shared__ __align__(16) double dg_smem[];
    if (P <= 3 && g.smr) dg_warp_strip<P, false, false, true, NEU, NoAcc>(g, chi, src, y, strip, j0, j1, nullptr, nullptr, dg_smem + (size_t)(threadIdx.x >> 5) * 5 * P * P * 32);
    else dg_warp_strip<P, false, false, false, NEU, NoAcc>(g, chi, src, y, strip, j0, j1, nullptr, nullptr, nullptr);
}

// ---- the CTA-tile kernel (fx_dgt.cuh): 2-D TMA staging, O(P) registers per thread -------------------------------------------
template <int P, bool NEU>
__global__ void __launch_bounds__(DgtCfg<P>::NT) __maxnreg__(DgtCfg<P>::REGS)
k_dgt_apply(const __grid_constant__ DgParams g, const __grid_constant__ DgtTile t, const __grid_constant__ CUtensorMap mu,
            const __grid_constant__ CUtensorMap muh, const __grid_constant__ CUtensorMap mc, const __grid_constant__ CUtensorMap mch,
            double* __restrict__ y) {
    extern __shared__ __align__(128) double dgt_smem[];
    __shared__ __align__(8) unsigned long long bars[DgtCfg<P>::NS];
    if (threadIdx.x == 0) {
        for (int s = 0; s < DgtCfg<P>::NS; ++s) fx_mbar_init(fx_smem_addr(bars) + 8u * s, 1u);
        fx_mbar_fence_init();
        fx_tma_prefetch_desc(&mu); fx_tma_prefetch_desc(&muh); fx_tma_prefetch_desc(&mc); fx_tma_prefetch_desc(&mch);
    }
    __syncthreads();
    const DgtDir nodir = {nullptr, nullptr, nullptr, 0.0, false};
    const int per = t.ntx * t.nseg, rem = (int)(blockIdx.x % per);
    dgt_tile<P, DgtCfg<P>::NBX, DgtCfg<P>::NS, false, false, NEU, NoAcc>(g, t, &mu, &muh, &mc, &mch, nodir, y, bars, rem % t.ntx, rem / t.ntx,
                                                                  (int)(blockIdx.x / per), nullptr, nullptr);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libfx.so does not link libcuda)
typedef CUresult (*fx_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static fx_encode_tiled_fn fx_encode_tiled() {
    static fx_encode_tiled_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            fn = (fx_encode_tiled_fn)p;
        tried = true;
    }
    return fn;
}

// tensor map over the row-major (rows x pitch) fp64 image at `base`, box = boxw x boxh doubles, zero fill outside
fx_status fx_dgt_make_map(CUtensorMap* m, const double* base, int pitch, int rows, int boxw, int boxh) {
    fx_encode_tiled_fn enc = fx_encode_tiled();
    if (!enc) { fx_set_error("cuTensorMapEncodeTiled is not available"); return FX_ECUDA; }
    const cuuint64_t dims[2] = {(cuuint64_t)pitch, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)pitch * 8ull};
    const cuuint32_t box[2] = {(cuuint32_t)boxw, (cuuint32_t)boxh};
    const cuuint32_t es[2] = {1u, 1u};
    const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, boxw >= 32 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_NONE,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { fx_set_error("cuTensorMapEncodeTiled failed (%d)", (int)r); return FX_ECUDA; }
    return FX_OK;
}

// The tile kernels need: even row pitch and 16-byte aligned images (TMA's global-memory rules), and cuTensorMapEncodeTiled.
bool fx_dgt_eligible(const fx_grid* g, const void* a, const void* b, const void* c2) {
    return ((g->Nx * g->P) & 1) == 0 && aligned16(a) && aligned16(b) && aligned16(c2) && fx_encode_tiled() != nullptr;
}

// Launch geometry: tiles of NBX blocks of wb <= 30 cells, balanced over the row; segments so that the grid is whole waves
// of `resident` CTAs with little prologue work (one extra cell row of loads and about half a row of arithmetic each).
void fx_dgt_shape(FxCtx* c, const fx_grid* g, int nbx, int resident, DgtTile* t, int Nz) {
    const int tmax = FX_STRIP * nbx;
    t->ntx = (g->Nx + tmax - 1) / tmax;
    t->wb = (g->Nx + t->ntx * nbx - 1) / (t->ntx * nbx);
    // every box must start on a 16-byte boundary of the image row (an odd starting column raised "illegal instruction" on
    // the B200): tiles start at even columns, i.e. an even number of doubles per tile; the one-cell halo boxes then start
    // at even columns too (fx_dgt.cuh, colL / colR)
    if ((t->wb * nbx * g->P) & 1) t->wb++;
    t->ntx = (g->Nx + t->wb * nbx - 1) / (t->wb * nbx);
    int rps = c->launch[2][0];
    if (rps <= 0) {
        double best = 1e300;
        rps = 1;
        for (int r = 1; r <= g->Ny; ++r) {
            const long long ctas = (long long)t->ntx * ((g->Ny + r - 1) / r) * Nz;
            const double cost = (double)((ctas + resident - 1) / resident) * (r + 1.0);
            if (cost <= best) { best = cost; rps = r; }
            if (ctas <= resident && r >= 2) break;
        }
    }
    if (rps > g->Ny) rps = g->Ny;
    t->rows_per_seg = rps;
    t->nseg = (g->Ny + rps - 1) / rps;
}

template <int P, bool NEU>
static fx_status launch_dgt_apply(FxCtx* c, const fx_grid* g, const DgParams& p, const double* chi, const double* x, double* y) {   // (p.Nz planes)
    constexpr int NBX = DgtCfg<P>::NBX;
    typedef DgtGeom<P, NBX, 2, DgtCfg<P>::NS> G;
    const int occ = fx_func_occ(c, (const void*)k_dgt_apply<P, NEU>, G::NT, G::SMEM, true);
    DgtTile t;
    fx_dgt_shape(c, g, NBX, c->num_sms * occ, &t, p.Nz);
    const int pitch = g->Nx * P, rows = g->Ny * P * p.Nz;
    CUtensorMap mu, muh, mc, mch;
    fx_status s;
    if ((s = fx_dgt_make_map(&mu, x, pitch, rows, G::BW, P)) != FX_OK || (s = fx_dgt_make_map(&muh, x, pitch, rows, G::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&mc, chi, pitch, rows, G::BW, P)) != FX_OK || (s = fx_dgt_make_map(&mch, chi, pitch, rows, G::HW, P)) != FX_OK)
        return s;
    k_dgt_apply<P, NEU><<<t.ntx * t.nseg * p.Nz, G::NT, G::SMEM, c->stream>>>(p, t, mu, muh, mc, mch, y);
    return FX_OK;
}

// a one-cell direction cannot carry a Dirichlet and a Neumann wall table at once (Q23)
static bool bc_ok(int bc, int N) { return bc >= FX_BC_PER && bc <= FX_BC_NEU_DIR && !(bc == FX_BC_DIR_NEU && N < 2); }
static int wall_lo(int bc) { return bc == FX_BC_PER ? 0 : (bc == FX_BC_DIR || bc == FX_BC_DIR_NEU) ? 1 : 2; }
static int wall_hi(int bc) { return bc == FX_BC_PER ? 0 : (bc == FX_BC_DIR || bc == FX_BC_NEU_DIR) ? 1 : 2; }
int fx_dg_has_neumann(const DgParams* p) { return p->lox == 2 || p->hix == 2 || p->loy == 2 || p->hiy == 2; }
// Which instantiation of the warp-strip kernels to launch.  The NEU = true one handles every wall kind; it is needed
// for Neumann walls and, at P = 4, preferred for all grids: ptxas allocates it without spills where the NEU = false one
// spills (apply at 1024^2: 110 us against 124 us).  Same arithmetic either way (the parity tests of P = 4 run through it).
int fx_dg_neu_variant(const DgParams* p, int P) { return fx_dg_has_neumann(p) || P == 4; }
int fx_grid_deriv_ok(const fx_grid* g) { return g->bcx <= FX_BC_DIR && g->bcy <= FX_BC_DIR; }

int fx_grid_ok(const fx_grid* g) {
    return g && g->Nx >= 1 && g->Ny >= 1 && g->P >= 1 && g->P <= FX_PMAX && g->lx > 0 && g->ly > 0 &&
           bc_ok(g->bcx, g->Nx) && bc_ok(g->bcy, g->Ny) &&
           (int64_t)g->Nx * g->P < (1ll << 30) && (int64_t)g->Ny * g->P < (1ll << 30);
}

// host scalars and tables exactly as DESIGN.md 3.4 writes them (plain IEEE double operations, no contraction)
fx_status fx_make_dg_params(const fx_grid* g, int normed, DgParams* o, double* vol4_out, int Nz, double lz) {
    fx_tables t;
    if (fx_make_tables(g->P, &t) != 0) { fx_set_error("P outside 1..5"); return FX_EINVAL; }
    memset(o, 0, sizeof(*o));
    const int P = g->P;
    volatile double hx = g->lx / g->Nx, hy = g->ly / g->Ny;
    volatile double hxhy = hx * hy;
    const double vol4 = hxhy / 4;
    o->Nx = g->Nx; o->Ny = g->Ny; o->bcx = g->bcx; o->bcy = g->bcy; o->normed = normed;
    // 3-D product grid (Q24): W3 = RN(hz*W2); the symmetric form is RN(hz*(S2 x)), the normed one is the plane's A2 x
    volatile double hz = lz > 0 ? lz / Nz : 1.0;
    const bool three_d = lz > 0;
    o->Nz = Nz > 0 ? Nz : 1; o->hz = hz; o->zmul = (three_d && !normed) ? 1 : 0;
    o->lox = wall_lo(g->bcx); o->hix = wall_hi(g->bcx); o->loy = wall_lo(g->bcy); o->hiy = wall_hi(g->bcy);
    o->cxx = hy / hx; o->cyy = hx / hy;
    volatile double hy2 = hy / 2, hx2 = hx / 2;
    for (int k = 0; k < P; ++k) {
        o->B[k] = t.B[k]; o->L[k] = t.L[k]; o->R[k] = t.R[k];
        o->JX[k] = hy2 * t.w[k]; o->JY[k] = hx2 * t.w[k];          // jump factor jf = 1 (Q8)
        for (int m = 0; m < P; ++m) {
            o->T0[k][m] = t.T0[k][m]; o->T0L[k][m] = t.T0L[k][m]; o->WW[k][m] = t.WW[k][m]; o->TD[k][m] = t.D[k][m];
            volatile double w = vol4 * t.WW[k][m];
            if (three_d && !normed) { volatile double w3 = hz * w; o->V[k][m] = 1.0 / w3; }      // preconditioner of the 3-D solve: V3 = 1/W3
            else o->V[k][m] = 1.0 / w;
        }
    }
    if (vol4_out) *vol4_out = vol4;
    return FX_OK;
}

// per-lane shared-memory row ring of the warp-strip kernels: 5 slots (8 with the fused direction update) of P*P doubles per lane
size_t fx_dg_ring_bytes(int P, int warps, bool dirf) { return (size_t)warps * (dirf ? 8 : 5) * P * P * 32 * sizeof(double); }

// Launch shape of the warp-strip kernels.  A warp = one strip of 30 cells x `rows_per_seg` cell rows; every segment pays
// a prologue of about 0.6 steps (the flux trace of the row below it).  Choose rows_per_seg to minimise
// waves * (rows_per_seg + 0.6), waves = ceil(warps / resident warps): whole waves, little redundant work, and for small
// grids as many warps as there are rows.
void fx_dg_shape(FxCtx* c, const fx_grid* g, DgParams* p, int warps_per_sm, int* grid, int* block, int max_wpb) {
    int wpb = c->launch[2][1] ? c->launch[2][1] / 32 : max_wpb;
    if (wpb > max_wpb) wpb = max_wpb;           // the kernels are compiled for <= 128 threads per CTA
    if (wpb < 1) wpb = 1;
    p->nstrip = (g->Nx + FX_STRIP - 1) / FX_STRIP;
    int rps = c->launch[2][0];
    if (rps <= 0) {
        const long long resident = (long long)c->num_sms * (warps_per_sm > 0 ? warps_per_sm : 12);
        double best = 1e300;
        rps = 1;
        for (int r = 1; r <= g->Ny; ++r) {
            const long long warps = (long long)p->nstrip * ((g->Ny + r - 1) / r) * (p->Nz > 0 ? p->Nz : 1);
            const double cost = (double)((warps + resident - 1) / resident) * (r + 0.6);
            if (cost <= best) { best = cost; rps = r; }
            if (warps <= resident && r >= 2) break;                   // one wave: larger segments only cost more
        }
    }
    if (rps > g->Ny) rps = g->Ny;
    p->rows_per_seg = rps;
    p->nseg = (g->Ny + rps - 1) / rps;
    const long long warps = (long long)p->nstrip * p->nseg * (p->Nz > 0 ? p->Nz : 1);
    *grid = (int)((warps + wpb - 1) / wpb);
    *block = wpb * 32;
}

fx_status fx_launch_apply(FxCtx* c, const fx_grid* g, const double* chi, const double* x, double* y, int normed, int Nz, double lz) {
    DgParams p;
    fx_status s = fx_make_dg_params(g, normed, &p, nullptr, Nz, lz);
    if (s != FX_OK) return s;
    const int neu = fx_dg_neu_variant(&p, g->P);
    int occw;                                                    // resident warps per SM of k_dg_apply<P, NEU>
    {
        const void* f;
        if (neu) f = g->P == 1 ? (const void*)k_dg_apply<1, true> : g->P == 2 ? (const void*)k_dg_apply<2, true> : g->P == 3 ? (const void*)k_dg_apply<3, true>
                   : g->P == 4 ? (const void*)k_dg_apply<4, true> : (const void*)k_dg_apply<5, true>;
        else f = g->P == 1 ? (const void*)k_dg_apply<1, false> : g->P == 2 ? (const void*)k_dg_apply<2, false> : g->P == 3 ? (const void*)k_dg_apply<3, false>
               : g->P == 4 ? (const void*)k_dg_apply<4, false> : (const void*)k_dg_apply<5, false>;
        const int w = g->P == 3 ? FX_AP_W : 4;
        occw = fx_func_occ(c, f, w * 32, 0) * w;
    }
    if (c->dg_path != 1 && fx_dgt_eligible(g, chi, x, y)) {
#define FX_TAPPLY(PP) \
    s = neu ? launch_dgt_apply<PP, true>(c, g, p, chi, x, y) : launch_dgt_apply<PP, false>(c, g, p, chi, x, y); break;
        const bool neu = fx_dg_has_neumann(&p) != 0;
        switch (g->P) {
        case 1: FX_TAPPLY(1)
        case 2: FX_TAPPLY(2)
        case 3: FX_TAPPLY(3)
        case 4: FX_TAPPLY(4)
        default: FX_TAPPLY(5)
        }
#undef FX_TAPPLY
        if (s != FX_OK) return s;
        c->launches++;
        FX_CUDA(cudaGetLastError());
        return FX_OK;
    }
    p.smr = 0;            // measured: the stand-alone apply is 2 % faster on the L1-prefetch path, the fused K1 6 % faster with the ring
    int grid, block;
    fx_dg_shape(c, g, &p, occw, &grid, &block, g->P == 3 ? FX_AP_W : 4);
    const size_t smem = p.smr ? fx_dg_ring_bytes(g->P, block / 32, false) : 0;
#define FX_APPLY(PP) \
    if (neu) k_dg_apply<PP, true><<<grid, block, smem, c->stream>>>(p, chi, x, y); \
    else k_dg_apply<PP, false><<<grid, block, smem, c->stream>>>(p, chi, x, y); \
    break;
    switch (g->P) {
    case 1: FX_APPLY(1)
    case 2: FX_APPLY(2)
    case 3: FX_APPLY(3)
    case 4: FX_APPLY(4)
    case 5: FX_APPLY(5)
    }
#undef FX_APPLY
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

static fx_status apply_checked(FxCtx* c, const fx_grid* g, const double* chi, const double* x, double* y, int normed) {
    FX_ENTER(c, "fx_dg_elliptic_apply");
    if (!fx_grid_ok(g) || !chi || !x || !y) { fx_set_error("fx_dg_elliptic_apply: bad grid or null pointer"); return FX_EINVAL; }
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    const double *ye = y + n;
    if ((x < ye && y < x + n) || (chi < ye && y < chi + n)) { fx_set_error("fx_dg_elliptic_apply: y overlaps an input"); return FX_EINVAL; }
    return fx_launch_apply(c, g, chi, x, y, normed);
}
extern "C" fx_status fx_dg_elliptic_apply_ex(fx_ctx* c, const fx_grid* g, const double* chi, const double* x, double* y) { return apply_checked(c, g, chi, x, y, 1); }
extern "C" fx_status fx_dg_elliptic_apply_sym_ex(fx_ctx* c, const fx_grid* g, const double* chi, const double* x, double* y) { return apply_checked(c, g, chi, x, y, 0); }
extern "C" fx_status fx_dg_elliptic_apply(const fx_grid* g, const double* chi, const double* x, double* y) {
    FxCtx* c = fx_default_ctx();
    return c ? apply_checked(c, g, chi, x, y, 1) : FX_ECUDA;
}
extern "C" fx_status fx_dg_elliptic_apply_sym(const fx_grid* g, const double* chi, const double* x, double* y) {
    FxCtx* c = fx_default_ctx();
    return c ? apply_checked(c, g, chi, x, y, 0) : FX_ECUDA;
}

// W[idx] = RN(vol4 * WW[l][k]),  V[idx] = RN(1 / W[idx])     (Fig. 2 "volume")
// 3-D product grid (hz3 != 0): W3 = RN(hz * W2) on every plane, V3 = RN(1 / W3) (Q24; g.V holds V3 then)
__global__ void k_dg_weights(const __grid_constant__ DgParams g, int P, double vol4, int hz3, double* W, double* V) {
    const long long pitch = (long long)g.Nx * P, n = pitch * g.Ny * P * g.Nz;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int l = (int)((i / pitch) % P), k = (int)((i % pitch) % P);
        if (W) { const double w = __dmul_rn(vol4, g.WW[l][k]); W[i] = hz3 ? __dmul_rn(g.hz, w) : w; }
        if (V) V[i] = g.V[l][k];
    }
}

fx_status fx_launch_weights(FxCtx* c, const fx_grid* g, double* W, double* V, int Nz, double lz) {
    DgParams p; double vol4;
    fx_status s = fx_make_dg_params(g, 0, &p, &vol4, Nz, lz);
    if (s != FX_OK) return s;
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P * p.Nz;
    int grid = (int)((n + 255) / 256); if (grid > c->num_sms * 32) grid = c->num_sms * 32;
    k_dg_weights<<<grid, 256, 0, c->stream>>>(p, g->P, vol4, lz > 0 ? 1 : 0, W, V);
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

extern "C" fx_status fx_dg_weights_ex(fx_ctx* c, const fx_grid* g, double* W, double* V) {
    FX_ENTER(c, "fx_dg_weights");
    if (!fx_grid_ok(g)) { fx_set_error("fx_dg_weights: bad grid"); return FX_EINVAL; }
    return fx_launch_weights(c, g, W, V, 1, 0.0);
}
extern "C" fx_status fx_dg_weights(const fx_grid* g, double* W, double* V) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_dg_weights_ex(c, g, W, V) : FX_ECUDA;
}

extern "C" fx_status fx_dg_tables(int32_t P, double* out) {
    fx_tables t;
    if (!out || fx_make_tables(P, &t) != 0) { fx_set_error("fx_dg_tables: bad arguments"); return FX_EINVAL; }
    double* o = out;
    for (int k = 0; k < P; ++k) *o++ = t.xi[k];
    for (int k = 0; k < P; ++k) *o++ = t.w[k];
    for (int k = 0; k < P; ++k) *o++ = t.L[k];
    for (int k = 0; k < P; ++k) *o++ = t.R[k];
    for (int k = 0; k < P; ++k) *o++ = t.B[k];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.T0[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.T0L[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.WW[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.D[k][m];
    return FX_OK;
}

// ------------------------------------------------------------------------------------------------------------
// timing hook (include/fx.h): average time of back-to-back calls, measured on the device
// ------------------------------------------------------------------------------------------------------------
// fp64 issue roof (SURVEY 8d "FP64 issue rate is a real second roof ... micro-benchmark it first"; the paper: "high number of
// 64-bit operations per memory load"): FX_ROOF_CHAINS independent dependent-FMA chains per thread, no memory traffic.
// One launch = num_sms * 8 CTAs x 256 threads x FX_ROOF_CHAINS x FX_ROOF_ITERS fused multiply-adds.
#define FX_ROOF_CHAINS 8
#define FX_ROOF_ITERS 4096
__global__ void __launch_bounds__(256) k_fp64_roof(double* out, double a, double b) {
    double v[FX_ROOF_CHAINS];
#pragma unroll
    for (int i = 0; i < FX_ROOF_CHAINS; ++i) v[i] = (double)(threadIdx.x + i);
#pragma unroll 1
    for (int it = 0; it < FX_ROOF_ITERS; it += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < FX_ROOF_CHAINS; ++i) v[i] = __fma_rn(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < FX_ROOF_CHAINS; ++i) s = __dadd_rn(s, v[i]);
    if (s == 12345.678) out[0] = s;                      // never true for the arguments used: keeps the chains alive
}

static fx_status time_one(FxCtx* c, int kind, const fx_grid* g, const double* a, const double* b, double* cc, int64_t n) {
    switch (kind) {
    case 14: k_fp64_roof<<<c->num_sms * 8, 256, 0, c->stream>>>(cc, 0.999999, 1e-9); c->launches++; return cudaGetLastError() == cudaSuccess ? FX_OK : FX_ECUDA;
    case 0: return fx_launch_exdot(c, a, b, n, c->result_dev);
    case 1: return fx_axpby_ex(c, 0.7, a, -0.3, cc, n);
    case 2: return fx_pointwise_dot_ex(c, 1.0, a, b, 0.0, cc, n);
    case 3: return fx_launch_apply(c, g, a, b, cc, 0);
    case 4: return fx_launch_apply(c, g, a, b, cc, 1);
    case 5: { double v; return fx_exdot_ex(c, a, b, n, &v, nullptr); }
    case 6: return fx_axpby_ex(c, 0.7, a, 1.0, cc, n);
    case 7: return launch_exdotn<3>(c, a, b, cc, n, c->result_dev);
    case 8: return fx_launch_exsum(c, a, n, c->result_dev);
    case 9: return fx_launch_derivative(c, g, 0, 0, 0.7, a, -0.3, cc);
    case 10: return fx_launch_derivative(c, g, 1, 0, 0.7, a, -0.3, cc);
    case 11: return fx_launch_derivative(c, g, 0, 2, 0.7, a, -0.3, cc);
    case 12: return fx_launch_derivative(c, g, 1, 2, 0.7, a, -0.3, cc);
    case 13: return fx_arakawa_ex(c, g, a, b, cc);
    }
    return FX_EINVAL;
}

extern "C" fx_status fx_time_primitive_ex(fx_ctx* c, int32_t kind, const fx_grid* g, const double* a, const double* b, double* cc, int64_t n,
                                       int32_t reps, double* ms_host) {
    FX_ENTER(c, "fx_time_primitive");
    if (kind < 0 || kind > 14 || n < 0 || reps < 1 || !ms_host || !a || !b || !cc) { fx_set_error("fx_time_primitive: bad arguments"); return FX_EINVAL; }
    if ((kind == 3 || kind == 4 || (kind >= 9 && kind <= 13)) && (!fx_grid_ok(g) || (int64_t)g->Nx * g->Ny * g->P * g->P != n)) { fx_set_error("fx_time_primitive: bad grid"); return FX_EINVAL; }
    cudaEvent_t e0, e1;
    FX_CUDA(cudaEventCreate(&e0)); FX_CUDA(cudaEventCreate(&e1));
    fx_status s = time_one(c, kind, g, a, b, cc, n);
    if (s == FX_OK) {
        cudaStreamSynchronize(c->stream);
        cudaEventRecord(e0, c->stream);
        for (int i = 0; i < reps && s == FX_OK; ++i) s = time_one(c, kind, g, a, b, cc, n);
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        *ms_host = (double)ms / reps;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return s;
}
extern "C" fx_status fx_time_primitive(int32_t kind, const fx_grid* g, const double* a, const double* b, double* cc, int64_t n,
                                       int32_t reps, double* ms_host) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_time_primitive_ex(c, kind, g, a, b, cc, n, reps, ms_host) : FX_ECUDA;
}

// ---- exact dot without any allocation (fx_exdot_static) ----------------------------------------------------------------
// For callers that may not call cudaMalloc (stream capture, serving loops): the long accumulator's device scratch is a
// file-scope array that every GPU loading the library holds until exit, instead of a context's work space.  One launch of
// the k_exdot kernel above, so n <= FX_EXDOT_STATIC_MAX_N (2^28: every 64-bit digit stays far from overflow in one launch).
// The array is shared by every call on the device and keeps the last call's contents: the part that must start at zero is
// cleared, stream-ordered, before the launch; two calls that overlap on the GPU (different streams) race on it.
#define FX_XS_WORDS (FX_NDIG + FX_NLIMB + 8 + 4)                    // digits, limbs, flags + ticket (64 B), census
static __device__ __align__(256) fx_u64 fx_exdot_static_scratch[FX_XS_WORDS];     // 1728 bytes

struct FxStaticDev { int state; fx_u64* base; int num_sms; int occ[2]; };          // state: 0 new, 1 ready, -1 failed
static FxStaticDev fx_xs_dev[64];
static std::mutex fx_xs_mu;

extern "C" fx_status fx_exdot_static(const double* x, const double* y, int64_t n, double* result_dev, void* stream) {
    if (n < 0 || (n > 0 && (!x || !y)) || !result_dev) { fx_set_error("fx_exdot_static: bad arguments"); return FX_EINVAL; }
    if (n > FX_EXDOT_STATIC_MAX_N) {
        fx_set_error("fx_exdot_static: n exceeds FX_EXDOT_STATIC_MAX_N (2^28 elements in one launch); use fx_exdot_async");
        return FX_EINVAL;
    }
    int dev = 0;
    FX_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { fx_set_error("fx_exdot_static: device ordinal beyond 63"); return FX_EINVAL; }
    const int bd = 256;
    const size_t smem = (size_t)EX_STAGES * 2 * EX_U * bd * sizeof(double);
    FxStaticDev* d = &fx_xs_dev[dev];
    {
        std::lock_guard<std::mutex> lk(fx_xs_mu);
        if (d->state == 0) {                   // set-up, once per device, with that device current
            d->state = -1;
            // in host code the array's name is a host-side stand-in: the device address comes from the runtime
            FX_CUDA(cudaGetSymbolAddress((void**)&d->base, fx_exdot_static_scratch));
            FX_CUDA(cudaDeviceGetAttribute(&d->num_sms, cudaDevAttrMultiProcessorCount, dev));
            const void* kf[2] = {(const void*)k_exdot<false, 0>, (const void*)k_exdot<true, 0>};
            for (int v = 0; v < 2; ++v) {
                FX_CUDA(cudaFuncSetAttribute(kf[v], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                FX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d->occ[v], kf[v], bd, smem));
                if (d->occ[v] < 1) { fx_set_error("fx_exdot_static: kernel does not fit an SM"); return FX_ECUDA; }
            }
            d->state = 1;
        }
        if (d->state != 1) { fx_set_error("fx_exdot_static: set-up failed on this device"); return FX_ECUDA; }
    }
    cudaStream_t st = (cudaStream_t)stream;
    ExGlobal g;
    g.dig = d->base;
    g.limbs = g.dig + FX_NDIG;
    g.flags = (int*)(g.limbs + FX_NLIMB);
    g.ticket = (unsigned int*)(g.flags + 4);
    g.stats = g.limbs + FX_NLIMB + 8;
    g.keep_limbs = 0;
    // digits, flags and ticket must be zero when the kernel starts (a finished launch leaves them so, an aborted one may not)
    FX_CUDA(cudaMemsetAsync(d->base, 0, FX_XS_WORDS * sizeof(fx_u64), st));
    const bool vec = aligned16(x) && aligned16(y);
    const long long tile = (long long)bd * EX_U;
    long long grid = ((long long)n + tile - 1) / tile;
    const long long gmax = (long long)d->num_sms * d->occ[vec ? 1 : 0];
    if (grid > gmax) grid = gmax;
    if (grid < 1) grid = 1;
    if (vec) k_exdot<true, 0><<<(int)grid, bd, smem, st>>>(x, y, (long long)n, g, 1, 1, result_dev);
    else k_exdot<false, 0><<<(int)grid, bd, smem, st>>>(x, y, (long long)n, g, 1, 1, result_dev);
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}
