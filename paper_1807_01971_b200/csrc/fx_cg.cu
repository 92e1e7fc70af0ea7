// fx_cg.cu -- preconditioned conjugate gradient (a Level-2 algorithm built from Level-1 calls only;
// the exact dot "is for example important in a conjugate gradient method").  Algorithm: DESIGN.md 3.5.
//
// Two drivers that produce bit-identical iterates:
//   * unfused: one kernel per primitive, both dot results visit the host every iteration -- the structure the paper
//     benchmarks (its GPU dot latency IS that host round trip);
//   * fused (default; the paper's remedy "fewer calls, fewer passes"): two kernels per iteration
//       K1  p = z + beta p formed on the fly from r and the previous p (z = V o r recomputed; p is double-buffered because
//           neighbouring warps still read the old one), q = S p, and the exact dot p.q accumulated while q is produced
//           -> alpha = rz / pq   (device)
//       K2  phi += alpha p;  r -= alpha q;  z = V o r on the fly;  exact dot r.z -> convergence test, beta (device)
//     11 vector passes instead of 19.  The scalars never leave the device; a `done` flag turns the kernels that
//     were enqueued past convergence into no-ops, and the host looks at it once per batch of iterations.

#include <math.h>
#include <type_traits>
#include <stdlib.h>
#include <string.h>

#include <cooperative_groups.h>

#include "fx_internal.h"
#include "fx_dgt.cuh"
#include "fx_stream.cuh"

namespace cgr = cooperative_groups;

struct CgScal {
    double rz, pq, alpha, beta, bz, thresh, dot;
    int done, status, iters, pad;
    double rzb[2];               // r.z entering iteration k (slot k & 1): written by K1(k), read by K2(k) and K1(k+1)
};

// The fused loop's reductions are finished by their consumers (fx_exdot.cuh, ex_publish / ex_fetch_round): K1(k) adds the
// digits of p.q to PQ[k & 1], every CTA of K2(k) rounds them and forms alpha; K2(k) adds r.z to RZ[k & 1], every CTA of
// K1(k+1) rounds them, tests convergence and forms beta.  A kernel pays no ticket, no last-CTA finaliser and no scalar
// round trip at its end (about 6 us per kernel, twice per iteration); the rounding at the start overlaps the first loads.
// CTA 0 re-zeroes the buffer of the iteration after next one kernel after its last reader finished.
struct CgRed {
    fx_u64* dig;                 // [4][FX_NDIG]: PQ[0], PQ[1], RZ[0], RZ[1]
    int* flags;                  // [4]
    fx_u64* stats;               // the context's slow-path census
    __device__ fx_u64* pq(int k) const { return dig + (size_t)(k & 1) * FX_NDIG; }
    __device__ fx_u64* rz(int k) const { return dig + (size_t)(2 + (k & 1)) * FX_NDIG; }
    __device__ int* pqf(int k) const { return flags + (k & 1); }
    __device__ int* rzf(int k) const { return flags + 2 + (k & 1); }
};

// start of K1(k): r.z of the previous iteration -> convergence test, beta.  Returns false if the loop is over.
__device__ __forceinline__ bool cg_k1_scalars(ExShared* sh, const CgRed& red, CgScal* sc, int k, double* beta) {
    double rzn;
    if (k == 0) rzn = sc->rzb[1];                                   // set up by the host: r.z of the start residual
    else rzn = ex_fetch_round(sh, red.rz(k - 1), red.rzf(k - 1));
    const bool lead = blockIdx.x == 0 && threadIdx.x == 0;
    if (k > 0 && __dsqrt_rn(rzn) <= sc->thresh) {
        if (lead) { sc->rz = rzn; sc->status = FX_OK; sc->iters = k; sc->done = 1; }
        return false;
    }
    *beta = k > 0 ? __ddiv_rn(rzn, sc->rzb[(k - 1) & 1]) : 0.0;
    if (lead) { sc->rzb[k & 1] = rzn; sc->rz = rzn; sc->iters = k + 1; }
    if (blockIdx.x == 0) {                                          // PQ of the next iteration: its last reader was K2(k-1)
        for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) red.pq(k + 1)[i] = 0ull;
        if (threadIdx.x == 0) *red.pqf(k + 1) = 0;
    }
    return true;
}
// start of K2(k): p.q -> breakdown test, alpha
__device__ __forceinline__ bool cg_k2_scalars(ExShared* sh, const CgRed& red, CgScal* sc, int k, double* alpha) {
    const double pq = ex_fetch_round(sh, red.pq(k), red.pqf(k));
    if (!(pq > 0.0) || isinf(pq)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) { sc->pq = pq; sc->status = FX_EBREAKDOWN; sc->done = 1; }
        return false;
    }
    *alpha = __ddiv_rn(sc->rzb[k & 1], pq);
    if (blockIdx.x == 0) {                                          // RZ of the next iteration: its last reader was K1(k)
        for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) red.rz(k + 1)[i] = 0ull;
        if (threadIdx.x == 0) { *red.rzf(k + 1) = 0; sc->pq = pq; sc->alpha = *alpha; }
    }
    return true;
}
// after the last enqueued iteration of a batch: r.z of iteration k -> rz, convergence (what K1(k+1) would find)
__global__ void __launch_bounds__(128) k_cg_finish(CgRed red, CgScal* sc, int k) {
    __shared__ ExShared sh;
    if (*(volatile int*)&sc->done) return;
    const double rzn = ex_fetch_round(&sh, red.rz(k), red.rzf(k));
    if (threadIdx.x == 0) {
        sc->rz = rzn; sc->dot = rzn;
        if (__dsqrt_rn(rzn) <= sc->thresh) { sc->status = FX_OK; sc->done = 1; }
    }
}

#define CG_K 4
#define CG_W 40
typedef ExAcc<CG_K, CG_W> CgAcc;
#ifndef FX_K1_K
#define FX_K1_K 4
#define FX_K1_WB 40
#define FX_K1_KL 0
#endif
typedef ExAcc<FX_K1_K, FX_K1_WB, FX_K1_KL> K1Acc;      // the accumulator of p.q inside the stencil kernel K1

// Programmatic dependent launch (optional, FX_PDL=1): K1 and K2 of the fused loop are launched with programmatic stream
// serialisation, so a kernel's CTAs are scheduled as soon as the previous kernel's CTAs leave the SMs, set up their
// shared memory and wait here until the previous kernel has completed and flushed; nothing that depends on it (not even
// the done flag) is read before, and nothing is written before.  Without the launch attribute both calls are no-ops.
// Measured on config 3: 196 us per iteration with it, 171 us without -- off by default.
#define FX_PDL_SYNC() cudaGridDependencySynchronize()
// ... and this is where a CTA lets the next kernel's CTAs be scheduled: after its main loop, so that they take over the SM
// as this kernel drains (round 1 triggered at the start: the next kernel's CTAs then sat on shared memory and registers for
// the whole kernel -- 196 us per iteration against 171 us)
#define FX_PDL_TRIGGER() cudaTriggerProgrammaticLaunchCompletion()

template <class... KArgs, class... Args>
static cudaError_t cg_launch(bool pdl, void (*kern)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ---- K1: direction update + apply + dot -------------------------------------------------------------------------
// Register budget of K1: __maxnreg__ instead of __launch_bounds__(threads, minBlocks) -- the latter makes
// ptxas pick 168 registers for anything between two and three 128-thread CTAs per SM, and K1<3> then spills 880 bytes;
// with the cap spelled out it needs 212 registers without spilling, 200 with 44 bytes.
#ifndef FX_K1_R
#define FX_K1_R 255      // registers per thread of K1<3>
#define FX_K1_W 4        // warps per CTA of K1<3>
#endif
#define K1_THREADS(P) ((P) == 3 ? FX_K1_W * 32 : 128)
template <int P, bool NEU>
__global__ void __maxnreg__(P <= 2 ? 128 : P == 3 ? FX_K1_R : 255)
k_cg_dir_apply_dot(const __grid_constant__ DgParams g, const double* __restrict__ chi, const double* __restrict__ pin,
                   const double* __restrict__ r, double* __restrict__ pout, double* __restrict__ q, CgRed red, CgScal* sc, int k) {
    __shared__ ExShared sh;
    FX_PDL_SYNC();
    if (*(volatile int*)&sc->done) return;
    const int wpb = blockDim.x >> 5;
    long long w = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    const long long per = (long long)g.nstrip * g.nseg;             // warps per plane (3-D product grid: planes stacked in the vectors)
    const bool mine = w < per * g.Nz;
    if (mine) {
        const long long zoff = (w / per) * ((long long)g.Nx * g.Ny * P * P);
        w %= per;
        chi += zoff; pin += zoff; r += zoff; pout += zoff; q += zoff;
    }
    if (mine) {                                                      // the warp's first rows on their way to L2 while beta is formed
        const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);
        int ci = strip * FX_STRIP - 1 + (threadIdx.x & 31);
        ci = ci < 0 ? 0 : ci >= g.Nx ? g.Nx - 1 : ci;
        const long long pitch = (long long)g.Nx * P;
        int j = seg * g.rows_per_seg - 1;
        if (j < 0) j = 0;
#pragma unroll
        for (int d = 0; d < 3; ++d, ++j) {
            if (j >= g.Ny) break;
            const long long off = (long long)j * P * pitch + (long long)ci * P;
#pragma unroll
            for (int l = 0; l < P; ++l) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(pin + off + l * pitch));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(chi + off + l * pitch));
                if (k > 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(r + off + l * pitch));
            }
        }
    }
    double beta;
    if (!cg_k1_scalars(&sh, red, sc, k, &beta)) return;
    ex_shared_init(&sh);
    K1Acc acc;
    acc.init();
    // first iteration: p = z was set up by the caller, copy it through; later: p = z + beta p
    const DgSrc src = {pin, r, pout, beta, k > 0};
    if (mine) {
        const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);
        const int j0 = seg * g.rows_per_seg;
        int j1 = j0 + g.rows_per_seg;
        if (j1 > g.Ny) j1 = g.Ny;
        extern __shared__ __align__(16) double dg_smem[];
        if (P <= 3 && g.smr) dg_warp_strip<P, true, true, true, NEU, K1Acc>(g, chi, src, q, strip, j0, j1, &acc, &sh, dg_smem + (size_t)(threadIdx.x >> 5) * 8 * P * P * 32);
        else dg_warp_strip<P, true, true, false, NEU, K1Acc>(g, chi, src, q, strip, j0, j1, &acc, &sh, nullptr);
    }
    FX_PDL_TRIGGER();
    acc.flush(&sh);
    ex_publish(&sh, red.pq(k), red.pqf(k), red.stats);
}

// K1 on the CTA-tile stencil (fx_dgt.cuh): rows of r, p_old and chi arrive by 2-D TMA, the direction update is formed in
// shared memory, q = S p leaves through coalesced stores and every (p, q) pair enters the column thread's exact-dot bins.
template <int P>
struct CgtCfg {
    static constexpr int NBX = P == 3 ? FX_K1T_NBX : DgtCfg<P>::NBX;      // x-blocks per tile
    static constexpr int ND = FX_K1T_ND;                                  // exact-dot warps per CTA
    static constexpr int NT = 32 * NBX * P + 32 * (ND > 0 ? ND : 0);
    static constexpr int MINB = P >= 4 ? 2 : 3;
    static constexpr int REGS = P == 3 ? FX_K1T_R : (65536 / (MINB * NT)) / 16 * 16 > 255 ? 255 : (65536 / (MINB * NT)) / 16 * 16;
};
template <int P, bool NEU>
__global__ void __launch_bounds__(CgtCfg<P>::NT) __maxnreg__(CgtCfg<P>::REGS)
k_cgt_dir_apply_dot(const __grid_constant__ DgParams g, const __grid_constant__ DgtTile t, const __grid_constant__ CUtensorMap mp,
                    const __grid_constant__ CUtensorMap mph, const __grid_constant__ CUtensorMap mc, const __grid_constant__ CUtensorMap mch,
                    const __grid_constant__ CUtensorMap mr, const __grid_constant__ CUtensorMap mrh, double* __restrict__ pout,
                    double* __restrict__ q, CgRed red, CgScal* sc, int k) {
    extern __shared__ __align__(128) double dgt_smem[];
    __shared__ ExShared sh;
    __shared__ __align__(8) unsigned long long bars[DGT_NS_K1];
    if (threadIdx.x == 0) {
        for (int s = 0; s < DGT_NS_K1; ++s) fx_mbar_init(fx_smem_addr(bars) + 8u * s, 1u);
        fx_mbar_fence_init();
        fx_tma_prefetch_desc(&mp); fx_tma_prefetch_desc(&mc); fx_tma_prefetch_desc(&mr);
    }
    __syncthreads();
    FX_PDL_SYNC();
    if (*(volatile int*)&sc->done) return;
    double beta;
    if (!cg_k1_scalars(&sh, red, sc, k, &beta)) return;
    ex_shared_init(&sh);
    CgAcc acc;
    acc.init();
    const DgtDir dir = {&mr, &mrh, pout, beta, k > 0};
    const int per = t.ntx * t.nseg, rem = (int)(blockIdx.x % per);
    dgt_tile<P, CgtCfg<P>::NBX, DGT_NS_K1, true, true, NEU, CgAcc, CgtCfg<P>::ND>(g, t, &mp, &mph, &mc, &mch, dir, q, bars, rem % t.ntx, rem / t.ntx,
                                                                                 (int)(blockIdx.x / per), &acc, &sh);
    FX_PDL_TRIGGER();
    acc.flush(&sh);
    ex_publish(&sh, red.pq(k), red.pqf(k), red.stats);
}

// launch state of the tile K1 for one solve: geometry and the tensor maps of p (both buffers), chi and r
struct CgTile {
    bool on;
    DgtTile t;
    int grid, block;
    size_t smem;
    CUtensorMap p[2], ph[2], c, ch, r, rh;
};

static CgTile* fx_cg_tile(FxCtx* c) {              // (tensor maps are 64-byte aligned objects: kept out of the stack frame)
    if (!c->cg_tile) c->cg_tile = aligned_alloc(64, (sizeof(CgTile) + 63) / 64 * 64);
    return (CgTile*)c->cg_tile;
}

template <int P, bool NEU>
static fx_status cgt_setup(FxCtx* c, const fx_grid* g, int Nz, const double* chi, const double* r, const double* pb0, const double* pb1, CgTile* ct) {
    constexpr int NBX = CgtCfg<P>::NBX;
    typedef DgtGeom<P, NBX, 3, DGT_NS_K1, CgtCfg<P>::ND> G;
    const int occ = fx_func_occ(c, (const void*)k_cgt_dir_apply_dot<P, NEU>, G::NT, G::SMEM, true);
    fx_dgt_shape(c, g, NBX, c->num_sms * occ, &ct->t, Nz);
    ct->grid = ct->t.ntx * ct->t.nseg * Nz; ct->block = G::NT; ct->smem = G::SMEM;
    const int pitch = g->Nx * P, rows = g->Ny * P * Nz;
    fx_status s;
    const double* pb[2] = {pb0, pb1};
    for (int i = 0; i < 2; ++i)
        if ((s = fx_dgt_make_map(&ct->p[i], pb[i], pitch, rows, G::BW, P)) != FX_OK || (s = fx_dgt_make_map(&ct->ph[i], pb[i], pitch, rows, G::HW, P)) != FX_OK) return s;
    if ((s = fx_dgt_make_map(&ct->c, chi, pitch, rows, G::BW, P)) != FX_OK || (s = fx_dgt_make_map(&ct->ch, chi, pitch, rows, G::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&ct->r, r, pitch, rows, G::BW, P)) != FX_OK || (s = fx_dgt_make_map(&ct->rh, r, pitch, rows, G::HW, P)) != FX_OK) return s;
    ct->on = true;
    return FX_OK;
}

// ---- K2 / K3: streaming kernels over (row, column block) chunks --------------------------------------------------
// A chunk is CG_U * blockDim.x consecutive columns of one image row, so that l = row % P is uniform and k = col % P
// is cheap; chunks are taken grid-stride and iterated incrementally (no division in the loop).
#define CG_U 2
struct ChunkIter {
    int row, cb, drow, dcb, cpr;
    __device__ __forceinline__ void init(long long c0, int grid, int cpr_) {
        cpr = cpr_; row = (int)(c0 / cpr_); cb = (int)(c0 - (long long)row * cpr_); drow = grid / cpr_; dcb = grid - drow * cpr_;
    }
    __device__ __forceinline__ void next() { row += drow; cb += dcb; if (cb >= cpr) { cb -= cpr; ++row; } }
};

template <int NA>
__device__ __forceinline__ void cg_issue(double* buf, int stage, const double* const (&arr)[NA], int pitch, int rows,
                                         const ChunkIter& it) {
    const int bd = blockDim.x;
    double* s0 = buf + (size_t)stage * NA * CG_U * bd;
    if (it.row < rows) {
        const long long base = (long long)it.row * pitch;
#pragma unroll
        for (int u = 0; u < CG_U; ++u) {
            const int slot = u * bd + threadIdx.x;
            const int col = it.cb * (CG_U * bd) + slot;
            const bool in = col < pitch;
            const long long e = in ? base + col : 0;
#pragma unroll
            for (int a = 0; a < NA; ++a) fx_cp_async8(fx_smem_addr(s0 + a * CG_U * bd + slot), arr[a] + e, in);
        }
    }
    fx_cp_commit();
}

// K2: phi += alpha p; r -= alpha q; z = V o r; dot(r, z)
template <int P>
__global__ void __launch_bounds__(256, 3) k_cg_update(const __grid_constant__ DgParams g, const double* __restrict__ p,
                                                      const double* __restrict__ q, double* phi, double* r, CgRed red,
                                                      CgScal* sc, int k) {
    extern __shared__ __align__(16) double cg_buf[];
    __shared__ ExShared sh;
    FX_PDL_SYNC();
    if (*(volatile int*)&sc->done) return;
    double alpha;
    if (!cg_k2_scalars(&sh, red, sc, k, &alpha)) return;
    const double nalpha = -alpha;
    ex_shared_init(&sh);
    CgAcc acc;
    acc.init();
    const int pitch = g.Nx * P, rows = g.Ny * P * g.Nz, bd = blockDim.x;
    const int cpr = (pitch + CG_U * bd - 1) / (CG_U * bd);
    const double* const arr[4] = {p, q, phi, r};
    ChunkIter iq, ic;
    iq.init(blockIdx.x, gridDim.x, cpr); ic = iq;
#pragma unroll
    for (int s = 0; s < FX_STAGES - 1; ++s) { cg_issue<4>(cg_buf, s, arr, pitch, rows, iq); iq.next(); }
    int stage = 0;
    for (; ic.row < rows; ic.next()) {
        int sq = stage + FX_STAGES - 1; if (sq >= FX_STAGES) sq -= FX_STAGES;
        cg_issue<4>(cg_buf, sq, arr, pitch, rows, iq); iq.next();
        fx_cp_wait<FX_STAGES - 1>();
        const double* s0 = cg_buf + (size_t)stage * 4 * CG_U * bd;
        FX_ASSERT(stage >= 0 && stage < FX_STAGES && ic.row >= 0 && ic.row < rows);
        const int l = ic.row % P;
        const long long base = (long long)ic.row * pitch;
        double rr[CG_U], zz[CG_U];
        bool act[CG_U];
#pragma unroll
        for (int u = 0; u < CG_U; ++u) {
            const int slot = u * bd + threadIdx.x;
            const int col = ic.cb * (CG_U * bd) + slot;
            act[u] = col < pitch;
            const double pv = s0[slot], qv = s0[CG_U * bd + slot], fv = s0[2 * CG_U * bd + slot], rv = s0[3 * CG_U * bd + slot];
            const double rn = __fma_rn(nalpha, qv, rv);                      // axpby(-alpha, q, 1, r)
            if (act[u]) {
                phi[base + col] = __fma_rn(alpha, pv, fv);                   // axpby(alpha, p, 1, phi)
                r[base + col] = rn;
            }
            rr[u] = act[u] ? rn : 0.0;
            zz[u] = act[u] ? __dmul_rn(g.V[l][col % P], rn) : 0.0;           // pointwise_dot(1, V, r, 0, z)
        }
        acc.add<CG_U>(rr, zz, act, &sh);
        if (++stage == FX_STAGES) stage = 0;
    }
    fx_cp_wait<0>();
    FX_PDL_TRIGGER();
    acc.flush(&sh);
    ex_publish(&sh, red.rz(k), red.rzf(k), red.stats);
}

// K2, fast path: all four vectors 16-byte aligned.  Linear tiles of 2*blockDim.x elements, one 16-byte vector per thread,
// array and tile.  The table indices l = row % P, k = col % P of a thread's elements are advanced incrementally from tile
// to tile (no division in the loop).
template <int P>
__device__ __forceinline__ void cg_update_pair(const DgParams& g, double alpha, double nalpha, int l, int k, int col, int pitch,
                                               const double2& pv, const double2& qv, const double2& fv, const double2& rv,
                                               double2& fo, double2& ro, double (&zz)[2]) {
    int k1 = k + 1, l1 = l;
    if (k1 == P) k1 = 0;
    if (col + 1 == pitch) { k1 = 0; l1 = l + 1; if (l1 == P) l1 = 0; }
    fo.x = __fma_rn(alpha, pv.x, fv.x); fo.y = __fma_rn(alpha, pv.y, fv.y);       // axpby(alpha, p, 1, phi)
    ro.x = __fma_rn(nalpha, qv.x, rv.x); ro.y = __fma_rn(nalpha, qv.y, rv.y);     // axpby(-alpha, q, 1, r)
    zz[0] = __dmul_rn(g.V[l][k], ro.x); zz[1] = __dmul_rn(g.V[l1][k1], ro.y);     // pointwise_dot(1, V, r, 0, z)
}

// The tiles are moved by TMA: one elected thread issues 1-D bulk copies (cp.async.bulk, UBLKCP in SASS) of the four vectors
// that complete on a `full` mbarrier; the warps release a stage through an `empty` mbarrier.  No per-thread copy
// instructions: the load/store-unit queue carries only the LDS.128 reads and the two STG.128 writes (the cp.async variant
// of round 1 stalled on mio_throttle).  K2_STAGES-1 tiles (48 KB) are in flight per CTA, three CTAs per SM.
#define K2_STAGES 4
template <int P>
__global__ void __launch_bounds__(256, 3) k_cg_update_tma(const __grid_constant__ DgParams g, const double* __restrict__ p,
                                                          const double* __restrict__ q, double* phi, double* r, CgRed red,
                                                          CgScal* sc, int kit) {
    extern __shared__ __align__(128) double cg_buf[];
    __shared__ ExShared sh;
    __shared__ __align__(8) unsigned long long bars[2 * K2_STAGES];
    const int pitch = g.Nx * P, bd = blockDim.x, nwarp = bd >> 5;
    const long long n = (long long)pitch * g.Ny * P * g.Nz;
    const long long tile = 2ll * bd, nfull = n / tile;
    const unsigned arr_bytes = 16u * bd, stage_bytes = 4u * arr_bytes;
    const unsigned sbase = fx_smem_addr(cg_buf), s0 = sbase + 16u * threadIdx.x;
    const unsigned full0 = fx_smem_addr(bars), empty0 = full0 + 8u * K2_STAGES;
    if (threadIdx.x == 0) {
        for (int s = 0; s < K2_STAGES; ++s) { fx_mbar_init(full0 + 8u * s, 1u); fx_mbar_init(empty0 + 8u * s, (unsigned)nwarp); }
        fx_mbar_fence_init();
    }
    __syncthreads();
    FX_PDL_SYNC();                          // barriers are set up while the previous kernel drains
    if (*(volatile int*)&sc->done) return;
    // my full tiles: blockIdx.x, +G, ...  (count as a 32-bit number)
    const int mine = blockIdx.x < nfull ? (int)((nfull - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;
    const long long step = (long long)gridDim.x * tile;
    auto issue = [&](int i) {                                         // thread 0: tile i of this CTA into stage i % K2_STAGES
        const int s = i % K2_STAGES;
        const long long e0 = ((long long)blockIdx.x + (long long)i * gridDim.x) * tile;
        const unsigned dst = sbase + s * stage_bytes, bar = full0 + 8u * s;
        FX_ASSERT(i >= 0 && i < mine && e0 >= 0 && e0 + tile <= n);      // a full tile of the vectors, a stage of the ring
        fx_mbar_expect_tx(bar, stage_bytes);
        fx_tma_load_1d(dst, p + e0, arr_bytes, bar);
        fx_tma_load_1d(dst + arr_bytes, q + e0, arr_bytes, bar);
        fx_tma_load_1d(dst + 2 * arr_bytes, phi + e0, arr_bytes, bar);
        fx_tma_load_1d(dst + 3 * arr_bytes, r + e0, arr_bytes, bar);
    };
    if (threadIdx.x == 0)
        for (int i = 0; i < K2_STAGES - 1 && i < mine; ++i) issue(i);
    // alpha from the digits K1 left (every CTA rounds them itself) while the first tiles are on their way
    double alpha;
    if (!cg_k2_scalars(&sh, red, sc, kit, &alpha)) {
        if (threadIdx.x == 0)                                        // (copies in flight into this CTA's shared memory must land first)
            for (int i = 0; i < K2_STAGES - 1 && i < mine; ++i) fx_mbar_wait(full0 + 8u * i, 0u);
        return;
    }
    const double nalpha = -alpha;
    ex_shared_init(&sh);
    CgAcc acc;
    acc.init();
    long long i0 = (long long)blockIdx.x * tile + 2 * threadIdx.x;
    int col = (int)(i0 % pitch), l = (int)((i0 / pitch) % P), k = col % P;
    const int dcol = (int)(step % pitch), dl = (int)((step / pitch) % P), dk1 = dcol % P, dk2 = ((dcol % P) - (pitch % P) + P) % P;
    double* of = phi + i0;
    double* orr = r + i0;
    for (int i = 0; i < mine; ++i) {
        const int s = i % K2_STAGES, use = i / K2_STAGES;
        if (threadIdx.x == 0 && i + K2_STAGES - 1 < mine) {          // refill the stage consumed in the previous iteration
            const int j = i + K2_STAGES - 1, sj = j % K2_STAGES, uj = j / K2_STAGES;
            if (uj > 0) fx_mbar_wait(empty0 + 8u * sj, (unsigned)((uj - 1) & 1));
            issue(j);
        }
        fx_mbar_wait(full0 + 8u * s, (unsigned)(use & 1));
        double2 pv, qv, fv, rv, fo, ro;
        const unsigned sa = s0 + s * stage_bytes;
        fx_lds128(pv, sa); fx_lds128(qv, sa + arr_bytes); fx_lds128(fv, sa + 2 * arr_bytes); fx_lds128(rv, sa + 3 * arr_bytes);
        double rr[2], zz[2];
        cg_update_pair<P>(g, alpha, nalpha, l, k, col, pitch, pv, qv, fv, rv, fo, ro, zz);
        __syncwarp();
        if ((threadIdx.x & 31) == 0) fx_mbar_arrive(empty0 + 8u * s);
        *reinterpret_cast<double2*>(of) = fo;
        *reinterpret_cast<double2*>(orr) = ro;
        rr[0] = ro.x; rr[1] = ro.y;
#ifndef FX_K2_NODOT
        acc.add_all<2>(rr, zz, &sh);
#endif
        of += step; orr += step;
        col += dcol;
        const bool wrapped = col >= pitch;
        col -= wrapped ? pitch : 0;
        k += wrapped ? dk2 : dk1; k -= (k >= P) ? P : 0;
        l += dl + (wrapped ? 1 : 0); l -= (l >= P) ? P : 0;
    }
    if (nfull * tile < n && (int)(nfull % gridDim.x) == (int)blockIdx.x) {   // the ragged tail tile: plain loads
        const long long e0 = nfull * tile + 2 * threadIdx.x;
        bool act[2] = {e0 < n, e0 + 1 < n};
        double rr[2] = {0.0, 0.0}, zz[2] = {0.0, 0.0};
#pragma unroll
        for (int u = 0; u < 2; ++u)
            if (act[u]) {
                const long long e = e0 + u;
                const int c0 = (int)(e % pitch), l0 = (int)((e / pitch) % P);
                phi[e] = __fma_rn(alpha, p[e], phi[e]);
                const double rnw = __fma_rn(nalpha, q[e], r[e]);
                r[e] = rnw;
                rr[u] = rnw; zz[u] = __dmul_rn(g.V[l0][c0 % P], rnw);
            }
        acc.add<2>(rr, zz, act, &sh);
    }
    FX_PDL_TRIGGER();
    acc.flush(&sh);
    ex_publish(&sh, red.rz(kit), red.rzf(kit), red.stats);
}

// ---- persistent driver for grids that fit in L2 --------------------------------------------------------
// One cooperative launch runs the whole loop: phase A (= K1) and phase B (= K2) of every iteration are separated by
// grid-wide exact reductions (ex_grid_reduce: one grid.sync each, every CTA rounds the merged digits itself), the
// scalars live in registers, nothing returns to the host until convergence.  Per iteration: two grid syncs instead of two
// launches, two single-pass tails and their gaps.  The arithmetic, and therefore every bit of the result, is unchanged.
// Digit buffers: pdig[0..1] for p.q of even/odd iterations, pdig[2..3] for r.z; CTA 0 re-zeroes the buffer of the next
// iteration one phase after its last reader has passed a grid sync.
template <int P, bool NEU>
__global__ void __launch_bounds__(128, 2)
k_cg_persistent(const __grid_constant__ DgParams g, const double* __restrict__ chi, double* r, double* p0, double* p1, double* q,
                double* phi, fx_u64* pdig, int* pflags, CgScal* sc, int maxit) {
    cgr::grid_group grid = cgr::this_grid();
    __shared__ ExShared sh;
    extern __shared__ __align__(16) double dg_smem[];
    const unsigned pitch = (unsigned)(g.Nx * P);
    const unsigned n = pitch * (unsigned)(g.Ny * P * g.Nz);          // the host takes this path only for n < 2^24
    const double thresh = sc->thresh;
    double rz = sc->rz, beta = 0.0;
    int status = FX_MAXIT, it;
    const int wpb = blockDim.x >> 5;
    const long long gw = (long long)blockIdx.x * wpb + (threadIdx.x >> 5), tw = (long long)gridDim.x * wpb;
    const long long per = (long long)g.nstrip * g.nseg, nwork = per * g.Nz;
    const long long n2 = (long long)g.Nx * g.Ny * P * P;
    const unsigned tile = blockDim.x * 2u, ntiles = (n + tile - 1) / tile;
    // phase B walks tiles blockIdx.x, +G, +2G, ...: a thread's two elements of a tile start at (col0, l0) and move by `step`
    const unsigned step = gridDim.x * tile, dcol = step % pitch;
    const int drow = (int)((step / pitch) % P);
    unsigned col0[2];
    int l0[2];
#pragma unroll
    for (int v = 0; v < 2; ++v) {
        const unsigned e = blockIdx.x * tile + (unsigned)v * blockDim.x + threadIdx.x;
        col0[v] = e % pitch; l0[v] = (int)((e / pitch) % P);
    }
    auto phaseB = [&](auto uu, const double alpha, const double nalpha, double* pout, CgAcc& acc) {
        constexpr int U = decltype(uu)::value;
        unsigned col[2] = {col0[0], col0[1]};
        int l[2] = {l0[0], l0[1]};
#pragma unroll 1
        for (unsigned t = blockIdx.x; t < ntiles; t += (unsigned)U * gridDim.x) {
            double pv[2 * U], qv[2 * U], fv[2 * U], rv[2 * U];
            unsigned ee[2 * U];
#pragma unroll
            for (int u = 0; u < 2 * U; ++u) {
                const unsigned tt = t + (unsigned)(u >> 1) * gridDim.x;
                ee[u] = tt < ntiles ? tt * tile + (unsigned)(u & 1) * blockDim.x + threadIdx.x : n;
                const bool in = ee[u] < n;
                pv[u] = in ? pout[ee[u]] : 0.0; qv[u] = in ? q[ee[u]] : 0.0; fv[u] = in ? phi[ee[u]] : 0.0; rv[u] = in ? r[ee[u]] : 0.0;
            }
#pragma unroll
            for (int h = 0; h < U; ++h) {
                double rr[2], zz[2];
                bool act[2];
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const int u = 2 * h + v;
                    const unsigned e = ee[u];
                    act[v] = e < n;
                    rr[v] = 0.0; zz[v] = 0.0;
                    if (act[v]) {
                        phi[e] = __fma_rn(alpha, pv[u], fv[u]);
                        const double rn = __fma_rn(nalpha, qv[u], rv[u]);
                        r[e] = rn;
                        rr[v] = rn; zz[v] = __dmul_rn(g.V[l[v]][col[v] % P], rn);
                    }
                    col[v] += dcol; l[v] += drow;                          // the same element of the next tile
                    if (col[v] >= pitch) { col[v] -= pitch; ++l[v]; }
                    if (l[v] >= P) l[v] -= P;
                    if (l[v] >= P) l[v] -= P;
                }
                acc.add<2>(rr, zz, act, &sh);
            }
        }
    };
#ifdef FX_PERSIST_PROF
    unsigned long long tp[5] = {0, 0, 0, 0, 0}, t0, t1;
#define FX_TICK(i) do { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); tp[i] += t1 - t0; t0 = t1; } while (0)
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
#else
#define FX_TICK(i)
#endif
    for (it = 1; it <= maxit; ++it) {
        const int k = it - 1;
        const double* pin = (k & 1) ? p1 : p0;
        double* pout = (k & 1) ? p0 : p1;
        // ---- phase A: p = z + beta p, q = S p, exact dot p.q ---------------------------------------------------------
        ex_shared_init(&sh);
        CgAcc acc;
        acc.init();
        {
            for (long long wz = gw; wz < nwork; wz += tw) {
                const long long zoff = (wz / per) * n2, w = wz % per;                      // 3-D product grid: this warp's plane
                const DgSrc src = {pin + zoff, r + zoff, pout + zoff, beta, k > 0};
                const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);
                const int j0 = seg * g.rows_per_seg;
                int j1 = j0 + g.rows_per_seg;
                if (j1 > g.Ny) j1 = g.Ny;
                // rows through the per-lane cp.async ring where it exists (P <= 3: the copies of the next step are in flight while this
                // one computes; cp.async.ca is an ordinary coherent access, unlike ld.global.nc), else coherent register loads
                if (P <= 3 && g.smr && g.rows_per_seg >= 2) dg_warp_strip<P, true, true, true, NEU, CgAcc, true>(g, chi + zoff, src, q + zoff, strip, j0, j1, &acc, &sh, dg_smem + (size_t)(threadIdx.x >> 5) * 8 * P * P * 32);
                else dg_warp_strip<P, true, true, false, NEU, CgAcc, true>(g, chi + zoff, src, q + zoff, strip, j0, j1, &acc, &sh, nullptr);
            }
        }
        acc.flush(&sh);
        FX_TICK(0);
        const double pq = ex_grid_reduce(&sh, pdig + (size_t)(k & 1) * FX_NDIG, pflags + (k & 1), grid);
        FX_TICK(1);
        if (blockIdx.x == 0) {
            for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) pdig[(size_t)((k + 1) & 1) * FX_NDIG + i] = 0ull;
            if (threadIdx.x == 0) pflags[(k + 1) & 1] = 0;
        }
        if (!(pq > 0.0) || isinf(pq)) { status = FX_EBREAKDOWN; break; }
        const double alpha = __ddiv_rn(rz, pq), nalpha = -alpha;
        // ---- phase B: phi += alpha p, r -= alpha q, z = V o r, exact dot r.z -----------------------------------------
        ex_shared_init(&sh);
        acc.init();
        // (the vectors sit in L2: a trip of this loop is one load round trip, so up to four tiles are fetched per trip; the table
        // indices of a thread's elements advance incrementally from tile to tile: no division in the loop)
        if (ntiles > gridDim.x) phaseB(std::integral_constant<int, 4>(), alpha, nalpha, pout, acc);
        else phaseB(std::integral_constant<int, 1>(), alpha, nalpha, pout, acc);
        acc.flush(&sh);
        FX_TICK(2);
        const double rzn = ex_grid_reduce(&sh, pdig + (size_t)(2 + (k & 1)) * FX_NDIG, pflags + 2 + (k & 1), grid);
        FX_TICK(3);
        if (blockIdx.x == 0) {
            for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) pdig[(size_t)(2 + ((k + 1) & 1)) * FX_NDIG + i] = 0ull;
            if (threadIdx.x == 0) pflags[2 + ((k + 1) & 1)] = 0;
        }
        if (__dsqrt_rn(rzn) <= thresh) { rz = rzn; status = FX_OK; break; }
        beta = __ddiv_rn(rzn, rz);
        rz = rzn;
    }
    if (it > maxit) it = maxit;
    if (blockIdx.x == 0 && threadIdx.x == 0) { sc->rz = rz; sc->status = status; sc->iters = it; sc->done = 1; }
#ifdef FX_PERSIST_PROF
    if (blockIdx.x == 0 && threadIdx.x == 0) printf("persistent: %d iterations, ns per iteration: phase A %.0f, reduce %.0f, phase B %.0f, reduce %.0f (grid %d)\n", it,
                                                    (double)tp[0] / it, (double)tp[1] / it, (double)tp[2] / it, (double)tp[3] / it, (int)gridDim.x);
#endif
}

template <int P, bool NEU>
static fx_status cg_run_persistent(FxCtx* c, const fx_grid* g, DgParams dp, const double* chi, double* r, double* p0, double* p1, double* q,
                                   double* phi, CgScal* sc, int maxit, bool* ran) {
    *ran = false;
    int coop = 0, occ = 0;
    FX_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device));
    if (!coop) return FX_OK;
    dp.smr = P <= 3 ? 1 : 0;
    const size_t psm = dp.smr ? fx_dg_ring_bytes(P, 4, true) : 0;
    occ = fx_func_occ(c, (const void*)k_cg_persistent<P, NEU>, 128, psm);
    FX_CUDA(cudaMemsetAsync(c->cg_pdig, 0, 4 * FX_NDIG * sizeof(fx_u64) + 64, c->stream));
    fx_u64* pdig = (fx_u64*)c->cg_pdig;
    int* pflags = (int*)(pdig + 4 * FX_NDIG);
    int ag, ab;
    fx_dg_shape(c, g, &dp, occ * 4, &ag, &ab);
    // as many CTAs as either phase can use, at most one resident wave (a cooperative launch must be co-resident)
    const long long n = (long long)g->Nx * g->Ny * g->P * g->P * dp.Nz;
    long long want = ((long long)dp.nstrip * dp.nseg * dp.Nz + 3) / 4, wantB = (n + 255) / 256;
    if (wantB > want) want = wantB;
    long long grid = (long long)c->num_sms * occ;
    if (want < grid) grid = want;
    if (grid < 1) grid = 1;
    void* args[] = {&dp, &chi, &r, &p0, &p1, &q, &phi, &pdig, &pflags, &sc, &maxit};
    FX_CUDA(cudaLaunchCooperativeKernel((const void*)k_cg_persistent<P, NEU>, dim3((unsigned)grid), dim3(128), args, psm, c->stream));
    c->launches++;
    *ran = true;
    return FX_OK;
}

// ------------------------------------------------------------------------------------------------------------

static fx_status cg_workspace(FxCtx* c, int64_t n) {
    if (c->cg_cap < n) {
        if (c->cg_vec) { cudaStreamSynchronize(c->stream); cudaFree(c->cg_vec); c->cg_vec = nullptr; c->cg_cap = 0; }
        if (cudaMalloc(&c->cg_vec, (size_t)8 * n * sizeof(double)) != cudaSuccess) {
            fx_set_error("CG work space: %s", cudaGetErrorString(cudaGetLastError())); return FX_ENOMEM;
        }
        c->cg_cap = n;
    }
    if (!c->cg_pdig) {                                            // digit buffers of the loop's reductions: PQ[2], RZ[2], flags
        if (cudaMalloc(&c->cg_pdig, 4 * FX_NDIG * sizeof(fx_u64) + 64) != cudaSuccess) { fx_set_error("CG digit buffers: %s", cudaGetErrorString(cudaGetLastError())); return FX_ENOMEM; }
    }
    if (!c->cg_scal) {
        if (cudaMalloc(&c->cg_scal, sizeof(CgScal)) != cudaSuccess || cudaMallocHost(&c->cg_scal_pinned, 2 * sizeof(CgScal)) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->cg_ev[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->cg_ev[1], cudaEventDisableTiming) != cudaSuccess) {
            fx_set_error("CG scalars: %s", cudaGetErrorString(cudaGetLastError())); return FX_ENOMEM;
        }
    }
    return FX_OK;
}

static void cg_shapes(FxCtx* c, const fx_grid* g, DgParams* p, int k1_warps_per_sm, int* apply_grid, int* apply_block, int* ew_grid, int* ew_block) {
    fx_dg_shape(c, g, p, k1_warps_per_sm, apply_grid, apply_block, K1_THREADS(g->P) / 32);
    int bd = c->launch[3][1] ? c->launch[3][1] : 256;
    if (bd > 256) bd = 256;
    const int pitch = g->Nx * g->P;
    const long long cpr = (pitch + (long long)bd * CG_U - 1) / ((long long)bd * CG_U);
    long long chunks = cpr * g->Ny * g->P * (p->Nz > 0 ? p->Nz : 1);
    long long gmax = (long long)c->num_sms * (768 / bd);           // one resident wave
    if (chunks > gmax) chunks = gmax;
    if (c->launch[3][0]) chunks = c->launch[3][0];
    *ew_grid = (int)chunks; *ew_block = bd;
}

template <int P>
static fx_status cg_enqueue_iters(FxCtx* c, const DgParams& dp, const CgTile& ct, int ag, int ab, int eg, int eb, const double* chi, double* phi,
                                  double* r, double* pbuf0, double* pbuf1, double* q, CgScal* sc, int first_index, int iters) {
    fx_func_occ(c, (const void*)k_cg_update<P>, 256, (size_t)FX_STAGES * 4 * CG_U * 256 * 8);
    fx_func_occ(c, (const void*)k_cg_update_tma<P>, 256, (size_t)K2_STAGES * 4 * 2 * 256 * 8);
    const size_t k1_smem = dp.smr ? fx_dg_ring_bytes(P, ab / 32, true) : 0;
    // K2 fast path: 16-byte aligned vectors (the work vectors always are; phi is the caller's)
    const bool lin = aligned16(phi) && aligned16(r) && aligned16(pbuf0) && aligned16(pbuf1) && aligned16(q);
    int lg;
    {
        const long long n = (long long)dp.Nx * dp.Ny * P * P * dp.Nz, tile = 2ll * eb;
        long long nt = (n + tile - 1) / tile, gm = (long long)c->num_sms * (768 / eb);
        if (nt > gm) nt = gm;
        if (c->launch[3][0]) nt = c->launch[3][0];
        lg = (int)nt;
    }
    const CgRed red = {(fx_u64*)c->cg_pdig, (int*)((fx_u64*)c->cg_pdig + 4 * FX_NDIG), c->ex.stats};
    for (int i = 0; i < iters; ++i) {
        // p is double-buffered: iteration k reads buffer k & 1 and writes the other one
        const int k = first_index + i;
        const double* pin = (k & 1) ? pbuf1 : pbuf0;
        double* pout = (k & 1) ? pbuf0 : pbuf1;
        cudaEvent_t* ev = nullptr;
        if (c->prof_on && k == 0) cudaEventRecord(c->prof_loop[0], c->stream);
        if (c->prof_on && k % c->prof_stride == 0 && c->prof_iters < c->prof_cap) { ev = c->prof_ev + 4 * c->prof_iters; c->prof_iters++; }
        if (ev) cudaEventRecord(ev[0], c->stream);
        const bool pdl = !ev && c->cg_pdl;                        // (profiling events between the kernels: plain launches)
        if (ct.on) {
            const int b = k & 1;
            if (fx_dg_has_neumann(&dp)) cg_launch(pdl, k_cgt_dir_apply_dot<P, true>, ct.grid, ct.block, ct.smem, c->stream, dp, ct.t, ct.p[b], ct.ph[b], ct.c, ct.ch, ct.r, ct.rh, pout, q, red, sc, k);
            else cg_launch(pdl, k_cgt_dir_apply_dot<P, false>, ct.grid, ct.block, ct.smem, c->stream, dp, ct.t, ct.p[b], ct.ph[b], ct.c, ct.ch, ct.r, ct.rh, pout, q, red, sc, k);
        } else if (fx_dg_neu_variant(&dp, P)) cg_launch(pdl, k_cg_dir_apply_dot<P, true>, ag, ab, k1_smem, c->stream, dp, chi, pin, r, pout, q, red, sc, k);
        else cg_launch(pdl, k_cg_dir_apply_dot<P, false>, ag, ab, k1_smem, c->stream, dp, chi, pin, r, pout, q, red, sc, k);
        if (ev) cudaEventRecord(ev[1], c->stream);
        if (lin) cg_launch(pdl, k_cg_update_tma<P>, lg, eb, (size_t)K2_STAGES * 4 * 2 * eb * 8, c->stream, dp, (const double*)pout, (const double*)q, phi, r, red, sc, k);
        else cg_launch(pdl, k_cg_update<P>, eg, eb, (size_t)FX_STAGES * 4 * CG_U * eb * 8, c->stream, dp, (const double*)pout, (const double*)q, phi, r, red, sc, k);
        if (ev) { cudaEventRecord(ev[2], c->stream); cudaEventRecord(ev[3], c->stream); }
        c->launches += 2;
    }
    if (c->prof_on) cudaEventRecord(c->prof_loop[1], c->stream);      // re-recorded after every batch: the last one stands
    if (iters > 0) {                                                  // r.z of the batch's last iteration -> rz, convergence, for the host
        k_cg_finish<<<1, 128, 0, c->stream>>>(red, sc, first_index + iters - 1);
        c->launches++;
    }
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

extern "C" fx_status fx_cg_profile_ex(fx_ctx* c, int32_t enable) {
    FX_ENTER(c, "fx_cg_profile");
    if (enable && !c->prof_ev) {
        c->prof_cap = 1024;
        c->prof_ev = (cudaEvent_t*)calloc((size_t)4 * c->prof_cap, sizeof(cudaEvent_t));
        for (int i = 0; i < 4 * c->prof_cap; ++i) FX_CUDA(cudaEventCreate(&c->prof_ev[i]));
        FX_CUDA(cudaEventCreate(&c->prof_loop[0]));
        FX_CUDA(cudaEventCreate(&c->prof_loop[1]));
    }
    c->prof_on = enable > 0 ? 1 : 0;
    c->prof_stride = enable > 0 ? enable : 1;
    return FX_OK;
}
extern "C" fx_status fx_cg_profile(int32_t enable) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_cg_profile_ex(c, enable) : FX_ECUDA;
}

extern "C" fx_status fx_cg_last_profile_ex(fx_ctx* c, double* ms, int32_t* iters) {
    FX_ENTER(c, "fx_cg_last_profile");
    if (!ms) { fx_set_error("fx_cg_last_profile: null pointer"); return FX_EINVAL; }
    for (int i = 0; i < 4; ++i) ms[i] = c->prof_ms[i];
    if (iters) *iters = c->prof_iters;
    return FX_OK;
}
extern "C" fx_status fx_cg_last_profile(double* ms, int32_t* iters) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_cg_last_profile_ex(c, ms, iters) : FX_ECUDA;
}

static fx_status cg_collect_profile(FxCtx* c, int iters_done) {
    for (int i = 0; i < 4; ++i) c->prof_ms[i] = 0.0;
    // sampled iterations: 0, stride, 2 stride, ... below iters_done
    int m = c->prof_iters;
    const int valid = iters_done > 0 ? (iters_done - 1) / c->prof_stride + 1 : 0;
    if (m > valid) m = valid;
    c->prof_iters = iters_done;
    if (m <= 0) return FX_OK;
    float t;
    FX_CUDA(cudaEventElapsedTime(&t, c->prof_loop[0], c->prof_loop[1]));
    c->prof_ms[0] = t;
    for (int i = 0; i < m; ++i)
        for (int k = 0; k < 3; ++k) {
            FX_CUDA(cudaEventElapsedTime(&t, c->prof_ev[4 * i + k], c->prof_ev[4 * i + k + 1]));
            c->prof_ms[1 + k] += t;
        }
    for (int k = 0; k < 3; ++k) c->prof_ms[1 + k] *= (double)iters_done / m;       // scaled from the m sampled iterations to the loop
    return FX_OK;
}

// The solve on Nz stacked planes of the grid g (Nz = 1, lz = 0: the 2-D solve; lz > 0: the 3-D product grid, Q24)
static fx_status cg_solve_impl(FxCtx* c, const fx_grid* g, int Nz, double lz, const double* chi, const double* rho, double* phi, double tol,
                               int32_t maxit, fx_cg_info* info) {
    if (!fx_grid_ok(g) || Nz < 1 || !chi || !rho || !phi || maxit < 0 || !(tol >= 0)) { fx_set_error("fx_cg_solve: bad arguments"); return FX_EINVAL; }
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P * Nz;
    if (n >= ((int64_t)1 << 31)) { fx_set_error("fx_cg_solve: more than 2^31 unknowns"); return FX_EINVAL; }
    fx_status s = cg_workspace(c, n);
    if (s != FX_OK) return s;
    double *W = c->cg_vec, *V = W + n, *rhs = V + n, *r = rhs + n, *z = r + n, *p = z + n, *q = p + n, *p2 = q + n;
    const size_t bytes = (size_t)n * sizeof(double);

    // setup with the public primitives (lines before the loop)
    if ((s = fx_launch_weights(c, g, W, V, Nz, lz)) != FX_OK) return s;
    if ((s = fx_pointwise_dot_ex(c, -1.0, W, rho, 0.0, rhs, n)) != FX_OK) return s;
    if ((s = fx_launch_apply(c, g, chi, phi, q, 0, Nz, lz)) != FX_OK) return s;
    FX_CUDA(cudaMemcpyAsync(r, rhs, bytes, cudaMemcpyDeviceToDevice, c->stream));
    if ((s = fx_axpby_ex(c, -1.0, q, 1.0, r, n)) != FX_OK) return s;
    if ((s = fx_pointwise_dot_ex(c, 1.0, V, rhs, 0.0, z, n)) != FX_OK) return s;
    double bz;
    if ((s = fx_exdot_ex(c, rhs, z, n, &bz, nullptr)) != FX_OK) return s;
    if (bz == 0.0) {
        FX_CUDA(cudaMemsetAsync(phi, 0, bytes, c->stream));
        FX_CUDA(cudaStreamSynchronize(c->stream));
        if (info) { info->iterations = 0; info->status = FX_OK; info->rel_residual = 0.0; }
        return FX_OK;
    }
    if ((s = fx_pointwise_dot_ex(c, 1.0, V, r, 0.0, z, n)) != FX_OK) return s;
    double rz;
    if ((s = fx_exdot_ex(c, r, z, n, &rz, nullptr)) != FX_OK) return s;
    FX_CUDA(cudaMemcpyAsync(p, z, bytes, cudaMemcpyDeviceToDevice, c->stream));
    const double thresh = tol * sqrt(bz);
    int it = 0, status = FX_OK;
    if (!(sqrt(rz) <= thresh)) {
        status = FX_MAXIT;
        if (!c->cg_fused) {
            for (it = 1; it <= maxit; ++it) {
                if ((s = fx_launch_apply(c, g, chi, p, q, 0, Nz, lz)) != FX_OK) return s;
                double pq;
                if ((s = fx_exdot_ex(c, p, q, n, &pq, nullptr)) != FX_OK) return s;
                if (!(pq > 0.0) || !isfinite(pq)) { status = FX_EBREAKDOWN; break; }
                const double alpha = rz / pq;
                if ((s = fx_axpby_ex(c, alpha, p, 1.0, phi, n)) != FX_OK) return s;
                if ((s = fx_axpby_ex(c, -alpha, q, 1.0, r, n)) != FX_OK) return s;
                if ((s = fx_pointwise_dot_ex(c, 1.0, V, r, 0.0, z, n)) != FX_OK) return s;
                double rz_new;
                if ((s = fx_exdot_ex(c, r, z, n, &rz_new, nullptr)) != FX_OK) return s;
                if (sqrt(rz_new) <= thresh) { rz = rz_new; status = FX_OK; break; }
                const double beta = rz_new / rz;
                if ((s = fx_axpby_ex(c, 1.0, z, beta, p, n)) != FX_OK) return s;
                rz = rz_new;
            }
            if (it > maxit) it = maxit;
        } else if (maxit > 0) {
            DgParams dp;
            if ((s = fx_make_dg_params(g, 0, &dp, nullptr, Nz, lz)) != FX_OK) return s;
            int ag, ab, eg, eb;
            int occb = 0;
            {
                const void* f;
                if (fx_dg_neu_variant(&dp, g->P))
                    f = g->P == 1 ? (const void*)k_cg_dir_apply_dot<1, true> : g->P == 2 ? (const void*)k_cg_dir_apply_dot<2, true>
                      : g->P == 3 ? (const void*)k_cg_dir_apply_dot<3, true> : g->P == 4 ? (const void*)k_cg_dir_apply_dot<4, true> : (const void*)k_cg_dir_apply_dot<5, true>;
                else
                    f = g->P == 1 ? (const void*)k_cg_dir_apply_dot<1, false> : g->P == 2 ? (const void*)k_cg_dir_apply_dot<2, false>
                      : g->P == 3 ? (const void*)k_cg_dir_apply_dot<3, false> : g->P == 4 ? (const void*)k_cg_dir_apply_dot<4, false> : (const void*)k_cg_dir_apply_dot<5, false>;
                dp.smr = g->P <= 3 ? 1 : 0;
                const int k1w = K1_THREADS(g->P) / 32;
                const size_t sm = dp.smr ? fx_dg_ring_bytes(g->P, k1w, true) : 0;
                occb = fx_func_occ(c, f, k1w * 32, sm) * k1w;
            }
            cg_shapes(c, g, &dp, occb > 0 ? occb : 4, &ag, &ab, &eg, &eb);
            if (!fx_cg_tile(c)) { fx_set_error("out of host memory"); return FX_ENOMEM; }
            CgTile& ct = *fx_cg_tile(c);
            ct.on = false;
            // K1 on the CTA-tile stencil: on request, and by default for P >= 4, where the warp-strip K1 spills (measured at 1024^2:
            // P = 4 326 against 368 us per iteration, P = 5 752 against 865; P = 2, 3: the strip K1 is faster)
            if ((c->dg_path == 2 || (c->dg_path == 0 && g->P >= 4)) && fx_dgt_eligible(g, chi, r, p) && aligned16(p2)) {
                const bool neu = fx_dg_has_neumann(&dp) != 0;
#define FX_CGT(PP) s = neu ? cgt_setup<PP, true>(c, g, Nz, chi, r, p, p2, &ct) : cgt_setup<PP, false>(c, g, Nz, chi, r, p, p2, &ct); break;
                switch (g->P) {
                case 1: FX_CGT(1)
                case 2: FX_CGT(2)
                case 3: FX_CGT(3)
                case 4: FX_CGT(4)
                default: FX_CGT(5)
                }
#undef FX_CGT
                if (s != FX_OK) return s;
            }
            CgScal* sc = (CgScal*)c->cg_scal;
            CgScal* hs = (CgScal*)c->cg_scal_pinned;
            memset(hs, 0, sizeof(*hs));
            hs->rz = rz; hs->bz = bz; hs->thresh = thresh; hs->status = FX_MAXIT;
            hs->rzb[1] = rz;                                     // K1(0) takes r.z of the start residual from here
            FX_CUDA(cudaMemcpyAsync(sc, hs, sizeof(CgScal), cudaMemcpyHostToDevice, c->stream));
            FX_CUDA(cudaMemsetAsync(c->cg_pdig, 0, 4 * FX_NDIG * sizeof(fx_u64) + 64, c->stream));
            FX_CUDA(cudaStreamSynchronize(c->stream));           // hs is reused as the read-back buffer
            // small grids (vectors resident in L2): the whole loop in one cooperative launch.  mode 1 = automatic,
            // 2 = never, 3 = whenever the device allows it (tests)
            bool persistent = false;
            if (((c->cg_fused == 1 && n <= ((int64_t)1 << 20)) || (c->cg_fused == 3 && n < ((int64_t)1 << 24)))) {
                const bool neuv = fx_dg_neu_variant(&dp, g->P) != 0;
                switch (g->P) {
                case 1: s = neuv ? cg_run_persistent<1, true>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent) : cg_run_persistent<1, false>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent); break;
                case 2: s = neuv ? cg_run_persistent<2, true>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent) : cg_run_persistent<2, false>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent); break;
                case 3: s = neuv ? cg_run_persistent<3, true>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent) : cg_run_persistent<3, false>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent); break;
                case 4: s = neuv ? cg_run_persistent<4, true>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent) : cg_run_persistent<4, false>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent); break;
                default: s = neuv ? cg_run_persistent<5, true>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent) : cg_run_persistent<5, false>(c, g, dp, chi, r, p, p2, q, phi, sc, maxit, &persistent); break;
                }
                if (s != FX_OK) return s;
                if (persistent) {
                    FX_CUDA(cudaMemcpyAsync(hs, sc, sizeof(CgScal), cudaMemcpyDeviceToHost, c->stream));
                    FX_CUDA(cudaStreamSynchronize(c->stream));
                    c->prof_iters = 0;
                }
            }
            // batches of iterations; the host looks at the `done` flag of batch b only after batch b+1 is enqueued,
            // so the device never idles while the flag travels
            CgScal* slot[2] = {hs, hs + 1};
            int enq = 0, batch = 8, nb = 0;
            bool finished = persistent;
            if (!persistent) c->prof_iters = 0;
            while (!finished) {
                if (enq < maxit) {
                    const int m = (maxit - enq < batch) ? (maxit - enq) : batch;
                    switch (g->P) {
                    case 1: s = cg_enqueue_iters<1>(c, dp, ct, ag, ab, eg, eb, chi, phi, r, p, p2, q, sc, enq, m); break;
                    case 2: s = cg_enqueue_iters<2>(c, dp, ct, ag, ab, eg, eb, chi, phi, r, p, p2, q, sc, enq, m); break;
                    case 3: s = cg_enqueue_iters<3>(c, dp, ct, ag, ab, eg, eb, chi, phi, r, p, p2, q, sc, enq, m); break;
                    case 4: s = cg_enqueue_iters<4>(c, dp, ct, ag, ab, eg, eb, chi, phi, r, p, p2, q, sc, enq, m); break;
                    default: s = cg_enqueue_iters<5>(c, dp, ct, ag, ab, eg, eb, chi, phi, r, p, p2, q, sc, enq, m); break;
                    }
                    if (s != FX_OK) return s;
                    enq += m;
                    FX_CUDA(cudaMemcpyAsync(slot[nb & 1], sc, sizeof(CgScal), cudaMemcpyDeviceToHost, c->stream));
                    FX_CUDA(cudaEventRecord(c->cg_ev[nb & 1], c->stream));
                    ++nb;
                    if (batch < 64) batch *= 2;
                    if (nb >= 2) {
                        FX_CUDA(cudaEventSynchronize(c->cg_ev[nb & 1]));         // the batch before the one just enqueued
                        if (slot[nb & 1]->done) finished = true;
                    }
                } else finished = true;
            }
            FX_CUDA(cudaStreamSynchronize(c->stream));
            if (!persistent) hs = slot[(nb - 1) & 1];                            // state after the last enqueued batch
            if (c->prof_on) { if ((s = cg_collect_profile(c, hs->iters)) != FX_OK) return s; }
            it = hs->iters; status = hs->status; rz = hs->rz;
        }
    }
    FX_CUDA(cudaStreamSynchronize(c->stream));
    if (info) { info->iterations = it; info->status = status; info->rel_residual = sqrt(rz) / sqrt(bz); }
    return (fx_status)status;
}
extern "C" fx_status fx_cg_solve_ex(fx_ctx* c, const fx_grid* g, const double* chi, const double* rho, double* phi, double tol, int32_t maxit,
                                    fx_cg_info* info) {
    FX_ENTER(c, "fx_cg_solve");
    return cg_solve_impl(c, g, 1, 0.0, chi, rho, phi, tol, maxit, info);
}
// 3-D product grid (fx.h; Q24)
static bool grid3_plane(const fx_grid3* g, fx_grid* p) {
    if (!g || g->Nz < 1 || !(g->lz > 0)) return false;
    p->Nx = g->Nx; p->Ny = g->Ny; p->P = g->P; p->lx = g->lx; p->ly = g->ly; p->bcx = g->bcx; p->bcy = g->bcy;
    return fx_grid_ok(p) != 0 && (int64_t)g->Ny * g->P * g->Nz < (1ll << 30);
}
extern "C" fx_status fx_cg3_solve_ex(fx_ctx* c, const fx_grid3* g, const double* chi, const double* rho, double* phi, double tol, int32_t maxit,
                                     fx_cg_info* info) {
    FX_ENTER(c, "fx_cg3_solve");
    fx_grid p;
    if (!grid3_plane(g, &p)) { fx_set_error("fx_cg3_solve: bad grid"); return FX_EINVAL; }
    return cg_solve_impl(c, &p, g->Nz, g->lz, chi, rho, phi, tol, maxit, info);
}
extern "C" fx_status fx_cg3_solve(const fx_grid3* g, const double* chi, const double* rho, double* phi, double tol, int32_t maxit, fx_cg_info* info) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_cg3_solve_ex(c, g, chi, rho, phi, tol, maxit, info) : FX_ECUDA;
}
extern "C" fx_status fx_dg3_elliptic_apply_ex(fx_ctx* c, const fx_grid3* g, const double* chi, const double* x, double* y, int32_t sym) {
    FX_ENTER(c, "fx_dg3_elliptic_apply");
    fx_grid p;
    if (!grid3_plane(g, &p) || !chi || !x || !y) { fx_set_error("fx_dg3_elliptic_apply: bad grid or null pointer"); return FX_EINVAL; }
    const int64_t n = (int64_t)p.Nx * p.Ny * p.P * p.P * g->Nz;
    if ((x < y + n && y < x + n) || (chi < y + n && y < chi + n)) { fx_set_error("fx_dg3_elliptic_apply: y overlaps an input"); return FX_EINVAL; }
    return fx_launch_apply(c, &p, chi, x, y, sym ? 0 : 1, g->Nz, g->lz);
}
extern "C" fx_status fx_dg3_elliptic_apply(const fx_grid3* g, const double* chi, const double* x, double* y, int32_t sym) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_dg3_elliptic_apply_ex(c, g, chi, x, y, sym) : FX_ECUDA;
}
extern "C" fx_status fx_dg3_weights_ex(fx_ctx* c, const fx_grid3* g, double* W, double* V) {
    FX_ENTER(c, "fx_dg3_weights");
    fx_grid p;
    if (!grid3_plane(g, &p)) { fx_set_error("fx_dg3_weights: bad grid"); return FX_EINVAL; }
    return fx_launch_weights(c, &p, W, V, g->Nz, g->lz);
}
extern "C" fx_status fx_dg3_weights(const fx_grid3* g, double* W, double* V) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_dg3_weights_ex(c, g, W, V) : FX_ECUDA;
}
extern "C" fx_status fx_cg_solve(const fx_grid* g, const double* chi, const double* rho, double* phi, double tol, int32_t maxit,
                                 fx_cg_info* info) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_cg_solve_ex(c, g, chi, rho, phi, tol, maxit, info) : FX_ECUDA;
}

// ---- host-buffer entry points (bench.py "e2e") ------------------------------------------------------------------

static fx_status stage_alloc(FxCtx* c, int64_t cap) {
    if (c->stage_cap < cap) {
        cudaStreamSynchronize(c->stream);
        for (int i = 0; i < 4; ++i) { if (c->stage[i]) cudaFree(c->stage[i]); c->stage[i] = nullptr; }
        c->stage_cap = 0;
        for (int i = 0; i < 4; ++i)
            if (cudaMalloc(&c->stage[i], (size_t)cap * sizeof(double)) != cudaSuccess) {
                fx_set_error("staging buffers: %s", cudaGetErrorString(cudaGetLastError())); return FX_ENOMEM;
            }
        c->stage_cap = cap;
    }
    if (!c->copy_stream) {
        FX_CUDA(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            FX_CUDA(cudaEventCreateWithFlags(&c->ev_copy[i], cudaEventDisableTiming));
            FX_CUDA(cudaEventCreateWithFlags(&c->ev_comp[i], cudaEventDisableTiming));
        }
    }
    return FX_OK;
}

extern "C" fx_status fx_cg_solve_host_ex(fx_ctx* c, const fx_grid* g, const double* chi, const double* rho, double* phi, double tol,
                                      int32_t maxit, fx_cg_info* info) {
    FX_ENTER(c, "fx_cg_solve_host");
    if (!fx_grid_ok(g) || !chi || !rho || !phi) { fx_set_error("fx_cg_solve_host: bad arguments"); return FX_EINVAL; }
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    fx_status s = stage_alloc(c, n);
    if (s != FX_OK) return s;
    const size_t bytes = (size_t)n * sizeof(double);
    FX_CUDA(cudaMemcpyAsync(c->stage[0], chi, bytes, cudaMemcpyHostToDevice, c->stream));
    FX_CUDA(cudaMemcpyAsync(c->stage[1], rho, bytes, cudaMemcpyHostToDevice, c->stream));
    FX_CUDA(cudaMemcpyAsync(c->stage[2], phi, bytes, cudaMemcpyHostToDevice, c->stream));
    s = fx_cg_solve_ex(c, g, c->stage[0], c->stage[1], c->stage[2], tol, maxit, info);
    if (s < 0) return s;
    FX_CUDA(cudaMemcpyAsync(phi, c->stage[2], bytes, cudaMemcpyDeviceToHost, c->stream));
    FX_CUDA(cudaStreamSynchronize(c->stream));
    return s;
}
extern "C" fx_status fx_cg_solve_host(const fx_grid* g, const double* chi, const double* rho, double* phi, double tol,
                                      int32_t maxit, fx_cg_info* info) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_cg_solve_host_ex(c, g, chi, rho, phi, tol, maxit, info) : FX_ECUDA;
}

// double-buffered: the copy of chunk i+1 overlaps the accumulation of chunk i
extern "C" fx_status fx_exdot_host_ex(fx_ctx* c, const double* x, const double* y, int64_t n, double* result_host) {
    FX_ENTER(c, "fx_exdot_host");
    if (n < 0 || (n > 0 && (!x || !y)) || !result_host) { fx_set_error("fx_exdot_host: bad arguments"); return FX_EINVAL; }
    const int64_t CH = (int64_t)1 << 23;                       // 64 MB per array and chunk
    fx_status s = stage_alloc(c, n < CH ? (n > 0 ? n : 1) : CH);
    if (s != FX_OK) return s;
    const int64_t cap = c->stage_cap < CH ? c->stage_cap : CH;
    const int64_t nch = n == 0 ? 1 : (n + cap - 1) / cap;
    cudaEventRecord(c->ev_comp[0], c->stream);
    cudaEventRecord(c->ev_comp[1], c->stream);
    for (int64_t i = 0; i < nch; ++i) {
        const int b = (int)(i & 1);
        const int64_t off = i * cap, m = (n - off < cap) ? (n - off) : cap;
        cudaStreamWaitEvent(c->copy_stream, c->ev_comp[b], 0);       // buffer b free again
        if (m > 0) {
            cudaMemcpyAsync(c->stage[2 * b], x + off, (size_t)m * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream);
            cudaMemcpyAsync(c->stage[2 * b + 1], y + off, (size_t)m * sizeof(double), cudaMemcpyHostToDevice, c->copy_stream);
        }
        cudaEventRecord(c->ev_copy[b], c->copy_stream);
        cudaStreamWaitEvent(c->stream, c->ev_copy[b], 0);
        if ((s = fx_launch_exdot_part(c, c->stage[2 * b], c->stage[2 * b + 1], m, i == 0, i == nch - 1, c->result_dev)) != FX_OK) return s;
        cudaEventRecord(c->ev_comp[b], c->stream);
    }
    return fx_result_to_host(c, result_host);
}
extern "C" double fx_exdot_host(const double* x, const double* y, int64_t n) {
    fx_set_error("%s", "");
    FxCtx* c = fx_default_ctx();
    if (!c) return NAN;
    double v = NAN;
    return fx_exdot_host_ex(c, x, y, n, &v) == FX_OK ? v : NAN;
}
